"""TEST INFRASTRUCTURE ONLY -- CPU oracle of the HARD-KV decode-step hot path.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  The product path (paper_2606_28831_b200) never does.
"""
