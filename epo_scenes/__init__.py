"""Seeded synthetic inputs shared by the oracle-side and CUDA-side tests and by bench.py.
Holds none of the EPO method's arithmetic (see generator.py)."""
from .generator import Scene, make_scene, CONFIGS, camera_centres, look_at, rodrigues, \
    rasterize_segments, render_depth_room, room_segments, all_directed_pairs, knn_pairs  # noqa: F401
from .rng import SplitMix64  # noqa: F401
