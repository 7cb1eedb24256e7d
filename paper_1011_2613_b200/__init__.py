"""paper_1011_2613_b200 -- B200-native LBM-IMB-DEM hot path (arxiv/paper_1011_2613).

`inputs`  : seeded synthetic workloads (shared with the tests' CPU oracle).
`binding` : thin ctypes binding of the C-ABI library include/lbmimb.h
            (csrc/*.cu, sm_100a); imported lazily so that `inputs` stays usable
            on a box without the built extension.
"""

__all__ = ["inputs", "binding"]
