"""B200-native mixed-precision CG solve of bond-network (pore / resistor network) Kirchhoff systems.

`inputs` (seeded synthetic networks) imports without CUDA; everything in `pn` needs the compiled
C-ABI library `libpn.so` (built by `paper_1908_03301_b200.build` / `__graft_entry__.build()`) and a
CUDA device -- there is no CPU fallback.
"""
__all__ = ["inputs", "pn", "build"]
