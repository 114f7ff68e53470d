"""Measurement and parity harness: seeded synthetic inputs (workloads.py, no method arithmetic) and the helpers that run
the CUDA library and the oracle on the same inputs (parity.py).  Neither product nor oracle: imported by tests/, bench.py
and __graft_entry__.smoke() only; the product package never imports it."""
