"""hard-b200: B200-native hot path of HARD (arxiv 2509.08971) — explicit finite-volume Euler update.

The CUDA library is loaded lazily by `paper_2509_08971_b200.hard`; importing the package (or
`paper_2509_08971_b200.workloads`) does not need a GPU or the built extension.
"""
