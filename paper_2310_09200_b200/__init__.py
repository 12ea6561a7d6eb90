"""B200-native Bluebild Standard Synthesizer (arXiv 2310.09200) — Python binding package.

``paper_2310_09200_b200.binding`` marshals arguments into the C-ABI library built from
``csrc/`` (every step of the path runs in CUDA kernels); ``workloads`` holds the seeded synthetic
inputs. Importing the package does not load the CUDA library; using the binding without it
raises loudly (there is no CPU fallback).
"""
__all__ = ["binding", "workloads"]
