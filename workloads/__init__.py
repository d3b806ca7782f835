"""Seeded synthetic workloads (input generators) for the TTS distillation step.

Serves both the oracle's tests and the CUDA path's tests / bench.py; holds none of the method's arithmetic and
imports neither ``oracle`` nor ``paper_2605_09329_b200``.
"""
