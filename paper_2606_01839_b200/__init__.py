"""conserve_kv: B200-native (sm_100a) KV-cache hot path of ConServe's conversation tail.

The product is the C-ABI library libconserve_kv.so (include/conserve_kv.h);
`paper_2606_01839_b200.binding` is a thin ctypes binding with the same names.
Importing this package does not load the library; the first call into
`binding` does, and fails loudly if it has not been built
(`python -c "import __graft_entry__ as g; g.build()"`).

`paper_2606_01839_b200.synth` (seeded input generators) has no dependency on
the library and none of the method's arithmetic.
"""
__version__ = "0.1.0"
