"""B200-native (sm_100a) data-parallel hot path of EMRI_MC (arXiv 2311.17174).

`paper_2311_17174_b200.emri` is the thin binding of the C-ABI library (include/emri.h);
`paper_2311_17174_b200.workloads` holds the seeded synthetic inputs.  Importing the package loads
nothing; `emri.load()` fails loudly when the CUDA library has not been built.
"""
__all__ = ["workloads", "emri"]
