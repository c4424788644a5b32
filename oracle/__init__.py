"""CPU oracle for the hot path of arxiv/paper_2511_08498 -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  The product (paper_2511_08498_b200) never does, and shares no code with it.
"""
