"""Bench-side microbenchmarks of the box (FP64 DFMA / DMMA rates, LDS.128 issue cost) that bench.py prints beside its
roofline.  Not part of the product: nothing under paper_2605_16734_b200/ imports this package, and libgcprobes.so is
built here, next to its source."""
