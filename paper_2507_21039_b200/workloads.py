"""Workload table of BASELINE.json's five configs (SURVEY.md 8(d) "Inputs") and of the Drell-Yan processes (8(f) f4).

This module holds NO arithmetic of the method: only process ids, seeds, batch sizes, energies and masses.
Both the CUDA path (through the C ABI) and the test oracle read their workload parameters from here; the
random numbers themselves come from each side's own Philox4x32-10, addressed by
(seed, global event index), so any sub-batch of a config is reproducible on either side.
"""
from collections import namedtuple

Workload = namedtuple("Workload", "cfg process name seed nevt sqrt_s final_masses precisions oracle_events")

MT = 173.0
# SM inputs: MZ, WZ, MT, WT, 1/alpha_EW, G_F, alpha_s  (BASELINE.json configs)
SM_PARAMS = (91.188, 2.441404, MT, 1.4915, 132.507, 1.16639e-5, 0.118)

WORKLOADS = {
    1: Workload(1, 1, "e+ e- -> mu+ mu-", 1, 16384, 500.0, (0.0, 0.0), ("d",), 16384),
    2: Workload(2, 2, "g g -> t t~", 2, 524288, 1500.0, (MT, MT), ("d", "f"), 524288),
    3: Workload(3, 3, "g g -> t t~ g", 3, 524288, 1500.0, (MT, MT, 0.0), ("d", "f", "m"), 524288),
    4: Workload(4, 4, "g g -> t t~ g g", 4, 262144, 1500.0, (MT, MT, 0.0, 0.0), ("d", "f"), 262144),
    5: Workload(5, 5, "g g -> t t~ g g g", 5, 65536, 1500.0, (MT, MT, 0.0, 0.0, 0.0), ("d", "f"), 2048),
    # the paper's other standard process, u u~ -> e+ e- + n g; not a BASELINE.json config.
    # Flat RAMBO without cuts like the others: soft and collinear gluons occur at their natural rate.
    6: Workload(6, 6, "u u~ -> e+ e-", 6, 524288, 1000.0, (0.0, 0.0), ("d", "f"), 524288),
    7: Workload(7, 7, "u u~ -> e+ e- g", 7, 524288, 1000.0, (0.0, 0.0, 0.0), ("d", "f"), 524288),
    8: Workload(8, 8, "u u~ -> e+ e- g g", 8, 262144, 1000.0, (0.0, 0.0, 0.0, 0.0), ("d", "f"), 262144),
    9: Workload(9, 9, "u u~ -> e+ e- g g g", 9, 65536, 1000.0, (0.0, 0.0, 0.0, 0.0, 0.0), ("d", "f"), 65536),
}

PRECISION_CODE = {"d": 0, "f": 1, "m": 2, "a": 3}      # a: all-FP32 (MG_FP32_ALL)
