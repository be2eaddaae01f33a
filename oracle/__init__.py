"""CPU oracle for the short-range force path.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this package.  It never imports paper_1410_2805_b200 and shares no code with it.
"""
