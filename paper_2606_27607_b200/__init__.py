"""B200-native phylogenetic-likelihood hot path (BEAGLE 4.1's method, arxiv/paper_2606_27607).

  plk        thin ctypes binding of the C-ABI library libplk.so (include/plk.h)
  client     drives a workload through the library the way a tree-inference package would (op lists from a tree)
  workloads  seeded synthetic inputs (BASELINE.json configs)
  build      in-tree nvcc build of libplk.so for sm_100a
"""
