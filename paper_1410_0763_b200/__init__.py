"""B200-native diffuse-radiation ray sweep (arXiv:1410.0763): thin Python binding over librt.so.

The binding only marshals arguments (torch tensors -> device pointers, streams); every step of the
path runs in the CUDA kernels of csrc/.  There is no CPU fallback: importing works without a GPU
(so that the build and the symbol table can be checked), but creating a context without a CUDA
device raises RtError.
"""
from .api import (RtError, RayTracer, healpix_dirs, load_library, rt_create, rt_destroy, rt_set_fields,  # noqa: F401
                  rt_set_inflow, rt_sweep, rt_segment_counts, rt_sum_ds, rt_total_segments,
                  rt_direction_records, rt_tune, RT_OWNED, RT_ATOMIC_ABLATION, RT_PAPER_GROUPS, RT_J_IN,
                  RT_J_TOTAL, RT_SUM_IN, rt_combine, rt_sweep_rates, rt_point_sources, rt_point_sources_static, RT_ELIMIT, RT_STATIC_MAX_SOURCES, RT_STATIC_MAX_BINS, rt_point_source_rates, rt_set_inflow_faces, rt_set_inflow_async, rt_set_inflow_faces_async, rt_debug_writer_counts, rt_working_set_bytes, rt_probe_bandwidth,
                  EXPORTED_SYMBOLS)
from .sharding import shard_directions, sweep_sharded, direction_work  # noqa: F401
