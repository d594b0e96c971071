"""Measurement / test harness code shared by tests/, bench.py and __graft_entry__.smoke(): seeded synthetic inputs only.
Not part of the product package and holds none of the method's arithmetic."""
