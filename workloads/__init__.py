"""Seeded synthetic workloads (inputs only; none of the method's arithmetic lives here)."""
