"""float64 CPU oracle of the TTT global-context-memory path — TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package. See oracle/ttt_oracle.c for the passages followed and the pins.
"""
