"""Pins for positions (Eq. 8 / 11) and the rotary delta correction (Eq. 9-10 / 12-13)."""
import numpy as np
import pytest

from helpers import read_fixture
from oracle import hermes_oracle as ho


def _cfg(d=16, **kw):
    base = dict(n_layers=1, n_q_heads=2, n_kv_heads=2, head_dim=d, budget=4, forget_rate=0.1,
                dtype="f32", rope_theta=10000.0)
    base.update(kw)
    return ho.OracleConfig(**base)


def _rope_ref(k0, pos_per_pair, theta):
    """Independent fp64 reference: RoPE as complex multiplication z_j * exp(i p theta_j)."""
    half = k0.shape[-1] // 2
    z = k0[..., :half].astype(np.float64) + 1j * k0[..., half:].astype(np.float64)
    z = z * np.exp(1j * pos_per_pair * theta)[:, None, :]
    return np.concatenate([z.real, z.imag], -1)


def test_hand_rotation_example():
    fx = read_fixture("hand_example.txt")
    cfg = _cfg(d=2, rope_theta=10000.0)                 # d = 2 -> theta_0 = 1 for any base
    k = fx["rot_in"].astype(np.float32).reshape(1, 1, 2)
    out = ho.rotary_delta(cfg, k, np.array([[-2]]))
    np.testing.assert_allclose(out.reshape(2), fx["rot_out"], atol=2e-6)   # sign or pair-layout slip fails


def test_frequencies_closed_form():
    th = ho.rope_frequencies(8, 10000.0)
    np.testing.assert_allclose(th, [1.0, 0.1, 0.01, 0.001], rtol=1e-14)


def test_rotation_composition_1d():
    cfg = _cfg(d=32, rope_theta=1.0e6)
    g = np.random.default_rng(0)
    n = 40
    k0 = g.standard_normal((n, 2, 32)).astype(np.float32)
    p = g.integers(0, 5000, n)
    q = g.integers(0, 5000, n)
    th = ho.rope_frequencies(32, cfg.rope_theta)
    k_p = _rope_ref(k0, p[:, None], th).astype(np.float32)
    k_q = _rope_ref(k0, q[:, None], th)
    out = ho.rotary_delta(cfg, k_p, (q - p)[None, :])
    # RoPE(k0,p) then delta(q-p) == RoPE(k0,q), to fp32 rounding of the pair norm
    half = 16
    nrm = np.hypot(k_q[..., :half], k_q[..., half:])
    err = np.abs(out - k_q)
    assert (err[..., :half] <= 4e-7 * nrm + 1e-30).all() and (err[..., half:] <= 4e-7 * nrm + 1e-30).all()


def test_rotation_norm_identity_inverse():
    cfg = _cfg(d=16)
    g = np.random.default_rng(1)
    k = g.standard_normal((9, 2, 16)).astype(np.float32)
    d0 = np.zeros((1, 9), np.int64)
    assert ho.rotary_delta(cfg, k, d0).tobytes() == k.tobytes()              # delta = 0: bit-exact copy
    dl = g.integers(-300, 0, (1, 9))
    out = ho.rotary_delta(cfg, k, dl)
    n_in = np.hypot(k[..., :8], k[..., 8:])
    n_out = np.hypot(out[..., :8], out[..., 8:])
    np.testing.assert_allclose(n_out, n_in, rtol=5e-7)                        # pair norm preserved
    back = ho.rotary_delta(cfg, out, -dl)
    np.testing.assert_allclose(back, k, atol=1e-6)                            # delta then -delta returns
    # mixed: only tokens with delta = 0 are bit-identical
    dl2 = dl.copy(); dl2[0, ::2] = 0
    out2 = ho.rotary_delta(cfg, k, dl2)
    assert out2[::2].tobytes() == k[::2].tobytes()
    assert not np.array_equal(out2[1::2], k[1::2])


def test_relative_position_invariance_pins_sign():
    # q.k depends only on (p_q - p_k): shift both by the same delta -> unchanged.  A wrong
    # rotation sign, or pairs (2j, 2j+1) instead of (j, j+d/2), breaks this.
    cfg = _cfg(d=32)
    g = np.random.default_rng(2)
    th = ho.rope_frequencies(32, cfg.rope_theta)
    q0 = g.standard_normal((1, 1, 32)).astype(np.float32)
    k0 = g.standard_normal((1, 1, 32)).astype(np.float32)
    qr = _rope_ref(q0, np.array([[900]]), th).astype(np.float32)
    kr = _rope_ref(k0, np.array([[700]]), th).astype(np.float32)
    before = float((qr.astype(np.float64) * kr).sum())
    q2 = ho.rotary_delta(cfg, qr, np.array([[-650]]))
    k2 = ho.rotary_delta(cfg, kr, np.array([[-650]]))
    after = float((q2.astype(np.float64) * k2).sum())
    assert after == pytest.approx(before, abs=2e-5)
    k_wrong = ho.rotary_delta(cfg, kr, np.array([[+650]]))
    assert abs(float((q2.astype(np.float64) * k_wrong).sum()) - before) > 1e-2


def test_mrope_sections_and_equivalence_to_1d():
    c3 = _cfg(d=128, rope_mode="m3d", mrope_section=(16, 24, 24), mrope_compact_axes=0b111)
    ax = ho.pair_axis(c3)
    assert (ax[:16] == 0).all() and (ax[16:40] == 1).all() and (ax[40:] == 2).all()
    c1 = _cfg(d=128)
    g = np.random.default_rng(3)
    k = g.standard_normal((7, 2, 128)).astype(np.float32)
    dl = g.integers(-50, 0, 7)
    a = ho.rotary_delta(c3, k, np.stack([dl, dl, dl]))
    b = ho.rotary_delta(c1, k, dl[None, :])
    assert a.tobytes() == b.tobytes()                      # t = h = w  ==  1D RoPE, same frequencies (c12)
    only_t = ho.rotary_delta(c3, k, np.stack([dl, 0 * dl, 0 * dl]))
    assert only_t[..., 16:64].tobytes() == k[..., 16:64].tobytes()       # h/w sections untouched
    assert only_t[..., 80:].tobytes() == k[..., 80:].tobytes()
    assert only_t[..., :16].tobytes() == b[..., :16].tobytes()


def test_bf16_rounding_is_rne():
    x = np.array([1.0, 1.0 + 2 ** -8, 1.0 + 3 * 2 ** -8, 1.0 + 2 ** -8 + 2 ** -20, -3.140625, 0.0], np.float32)
    r = ho.round_to_storage(x, "bf16")
    np.testing.assert_array_equal(r, np.array([1.0, 1.0, 1.0 + 2 ** -6, 1.0 + 2 ** -7, -3.140625, 0.0], np.float32))
    import torch
    y = np.random.default_rng(0).standard_normal(4096).astype(np.float32) * 37
    np.testing.assert_array_equal(ho.round_to_storage(y, "bf16"),
                                  torch.from_numpy(y).bfloat16().float().numpy())   # library RNE


def test_compact_positions_1d_and_m3d():
    c = _cfg(pos_offset=13)
    p = np.array([[13, 17, 18, 40, 41]])
    assert ho.compact_positions(c, p)[0].tolist() == [13, 14, 15, 16, 17]
    c3 = _cfg(d=128, rope_mode="m3d", mrope_compact_axes=0b001, pos_offset=2)
    pos = np.array([[5, 5, 9, 9, 9, 30], [2, 3, 2, 4, 9, 2], [7, 2, 2, 3, 3, 9]])
    out = ho.compact_positions(c3, pos)
    assert out[0].tolist() == [2, 2, 3, 3, 3, 4]           # distinct t's -> contiguous ranks, order kept
    assert out[1].tolist() == pos[1].tolist() and out[2].tolist() == pos[2].tolist()   # h/w preserved
    c3all = _cfg(d=128, rope_mode="m3d", mrope_compact_axes=0b111, pos_offset=2)
    out = ho.compact_positions(c3all, pos)
    assert out[1].tolist() == [2, 3, 2, 4, 5, 2] and out[2].tolist() == [4, 2, 2, 3, 3, 5]
    assert (out <= pos).all()                              # left-compaction never moves right
