"""B200-native MANTA vehicle-update hot path (arxiv 2007.03614): C-ABI library libmanta.so + thin binding.

    from paper_2007_03614_b200 import binding, workloads
    sim = binding.Sim(net, params, trips)      # manta_create + manta_load_trips
    sim.step(7200)                             # the hot path: manta_step
    out = sim.readback()                       # manta_readback
"""
__all__ = ["binding", "workloads", "build"]
