"""Measurement probes behind the roofline statements of DESIGN.md (run: python -m paper_2606_21023_b200.probes)."""
