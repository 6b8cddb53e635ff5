"""Measurement-only code that is NOT part of libbd: the FP64 issue-rate microbenchmark that gives bench.py its
roofline denominator (MEASURED_PEAKS.json carries no FP64 number)."""
