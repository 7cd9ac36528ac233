"""Test-support modules shared by tests/, bench.py and __graft_entry__.smoke(): the seeded synthetic input generator
(workloads.py).  Nothing here is part of the shipped package and nothing here scores a plan."""
