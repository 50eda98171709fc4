"""B200-native HLT1 Downstream + ghost-killer MLP + two-track vertexing (arXiv:2503.13092): libds and its binding."""
from .ds import (Downstream, DsError, ds_clone_kill, ds_create, ds_destroy, ds_error_string, ds_extrapolate, ds_ghost_killer,  # noqa: F401
                 ds_layout, ds_lines, ds_measure_dfma_peak, ds_process_host, ds_profile_enable, ds_profile_read, ds_reconstruct, ds_upload_geometry, ds_upload_line_nets, ds_upload_mlp_single, ds_version, ds_vertex, ds_vertex_static, ds_vertex_static_setup,
                 ds_vertex_workspace_bytes, ds_workspace_bytes, host_tracks, host_vertices, lib, make_geometry,
                 make_mlp, make_params)
