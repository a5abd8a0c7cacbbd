"""B200-native (sm_100a) hot path of the modified planar rotator (MPR)
conditional simulation (arXiv 1811.01604): checkerboard hybrid Monte Carlo
sweep, equilibration, M realizations, back-transform.

`paper_1811_01604_b200.mpr`   - thin Python binding of the C-ABI library
                                (include/mpr.h); argument marshalling only.
`paper_1811_01604_b200.synth` - seeded synthetic inputs and scores (none of the sweep's arithmetic; `choose_T`,
  the input temperature, restates Eq. 1 / Eq. 4 / reading R15 and is checked against the oracle in the tests).
`paper_1811_01604_b200.build` - compiles csrc/*.cu in-tree for sm_100a.

Nothing here imports `oracle/` and there is no CPU fallback: every call into
`mpr` fails loudly if the CUDA library is missing.
"""

__all__ = ["mpr", "synth", "build"]
