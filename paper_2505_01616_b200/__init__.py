"""phs -- B200-native batched flow-level network simulator (the netsim hot path of arxiv 2505.01616).

`paper_2505_01616_b200.binding` is the thin ctypes binding of the C-ABI library (include/phs.h);
`paper_2505_01616_b200.workloads` holds the seeded synthetic input generators (no method arithmetic).
Importing the package loads nothing native; the binding loads libphs.so on first use and fails loudly
if it is missing.
"""
__all__ = ["binding", "workloads"]
