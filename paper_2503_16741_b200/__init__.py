"""B200-native separable-footprint (SF-TR) X-ray projector pair: ct_fp_sf / ct_bp_sf behind a C ABI.

    from paper_2503_16741_b200 import binding      # ct_geom_create, ct_fp_sf, ct_bp_sf, ct_geom_destroy
    from paper_2503_16741_b200.projector import Geometry, Projector, FP, BP
    from paper_2503_16741_b200 import workloads    # seeded synthetic inputs (no method arithmetic)

The CUDA library is built in-tree by `python -m paper_2503_16741_b200.build`; there is no CPU fallback.
"""
__all__ = ["binding", "projector", "workloads", "geometry", "build"]
