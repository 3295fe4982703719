"""vog -- B200-native hot path of the 1Dx1D semi-Lagrangian Vlasov-Poisson solver of
arXiv 1301.5892 ("Vlasov on GPU").  The product is the C-ABI library built from
csrc/ (declared in include/vog.h); `vog` is its thin ctypes binding, `inputs` the
seeded workload generators.  Nothing here falls back to a CPU path."""
