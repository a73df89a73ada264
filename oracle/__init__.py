"""CPU oracle package.  TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke()
and bench.py's cpu_baseline / --impl reference legs; never from paper_2601_14724_b200/."""
