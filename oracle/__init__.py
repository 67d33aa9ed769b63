"""TEST INFRASTRUCTURE -- the fp64 CPU oracle written from PAPER.md (see hyb_oracle.h).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It shares nothing with paper_1406_6158_b200/.
"""
