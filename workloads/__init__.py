"""Seeded synthetic input generators and neutral workload descriptions (no method arithmetic).

Serves both the CUDA-path harness and the oracle harness; imports neither.
"""
