"""Seeded synthetic inputs for the cache-line collective simulator.

This package only BUILDS inputs (topologies as CSR, collective step DAGs, GPU
parameter sets, design-point lists).  It holds none of the simulation method's
arithmetic: no routing, no timing, no queueing.  Both the CPU oracle
(`oracle/`) and the CUDA engine (`paper_2606_10440_b200/`) receive the arrays
produced here, byte for byte; neither imports the other.

Shapes follow BASELINE.json `configs` and SURVEY.md section 8(d); the paper's
own workloads are synthetic collectives on a generic power-of-two GPU
 and ship no data, so these stand in for them.
"""
from .types import Topology, Collective, GpuCfg, Workload, DEP_DELIVERED, DEP_ACKED, DEP_ISSUED
from .rng import SplitMix64, config_seed
from . import topologies, collectives, configs, noc

__all__ = [
    "Topology", "Collective", "GpuCfg", "Workload",
    "DEP_DELIVERED", "DEP_ACKED", "DEP_ISSUED",
    "SplitMix64", "config_seed", "topologies", "collectives", "configs", "noc",
]
