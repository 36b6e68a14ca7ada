"""CPU oracle for cross-mesh resharding (arXiv 2211.05322) -- TEST INFRASTRUCTURE ONLY.

data_oracle : ctypes front end of reshard_oracle.c (the data result)
plan_oracle : unit tasks (App. B.2) and sender choice (Eq. 4), pure Python, tiny inputs

Nothing under paper_2211_05322_b200/ imports this package and this package imports nothing
from it.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may use it.
"""
