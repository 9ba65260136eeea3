"""B200-native batched goodput estimation for deployment-plan search (arxiv/paper_2512_14098).

`paper_2512_14098_b200.binding` is the thin ctypes binding of the C ABI in include/cf.h (imports
torch and loads libcf_b200.so; fails loudly if the library is missing). `workloads` holds the seeded
synthetic input generators and imports neither the binding nor the oracle.
"""
