"""CPU oracle for the Odyssey hot path — TEST INFRASTRUCTURE (see odyssey_oracle.cpp's header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It never imports paper_1601_02063_b200.
"""
