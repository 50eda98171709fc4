"""The C ABI without a GPU: the header is plain C, libds.so builds for sm_100a, loads, exports every function that
include/ds.h declares, the ctypes structs have the C sizes, and the product path fails loudly without a device."""
import ctypes as ct
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "ds.h")


def declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ds_[a-z_]+)\s*\(", src)))


def test_exports_every_declared_symbol():
    import paper_2503_13092_b200 as pk
    L = pk.lib()
    names = declared_functions()
    assert {"ds_create", "ds_destroy", "ds_upload_geometry", "ds_layout", "ds_extrapolate", "ds_reconstruct",
            "ds_ghost_killer", "ds_clone_kill", "ds_upload_line_nets", "ds_upload_mlp_single", "ds_lines", "ds_vertex", "ds_process_host", "ds_workspace_bytes", "ds_vertex_workspace_bytes",
            "ds_profile_enable", "ds_profile_read", "ds_measure_dfma_peak", "ds_kernel_name", "ds_error_string", "ds_version"} <= set(names)
    for n in names:
        assert hasattr(L, n), n
        assert hasattr(pk, n) or n in ("ds_kernel_name",), f"binding lacks {n}"


def test_header_is_plain_c_and_struct_sizes_match(tmp_path):
    import paper_2503_13092_b200.ds as B
    prog = tmp_path / "sz.c"
    prog.write_text('#include <stdio.h>\n#include "ds.h"\nint main(void){printf("%zu %zu %zu %zu %zu %zu %zu %zu %zu %zu %zu\\n",'
                    "sizeof(ds_geometry),sizeof(ds_mlp),sizeof(ds_params),sizeof(ds_hits),sizeof(ds_seeds),"
                    "sizeof(ds_tracks),sizeof(ds_vertices),sizeof(ds_layout_out),sizeof(ds_profile),sizeof(ds_mlp_single),"
                    "sizeof(ds_line_nets));return 0;}\n")
    exe = tmp_path / "sz"
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Wextra", "-Werror", "-pedantic", "-I", os.path.join(ROOT, "include"),
                    "-o", str(exe), str(prog)], check=True)
    sizes = [int(x) for x in subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.split()]
    mine = [ct.sizeof(t) for t in (B.DsGeometry, B.DsMlp, B.DsParams, B.DsHits, B.DsSeeds, B.DsTracks, B.DsVertices,
                                   B.DsLayoutOut, B.DsProfile, B.DsMlpSingle, B.DsLineNets)]
    assert sizes == mine


def test_cuda_sources_target_sm100a_only():
    import paper_2503_13092_b200.build as bld
    assert "arch=compute_100a,code=sm_100a" in bld.NVCC_FLAGS and "-lineinfo" in bld.NVCC_FLAGS
    out = subprocess.run(["cuobjdump", "-lelf", bld.build()], capture_output=True, text=True).stdout
    assert "sm_100a" in out and not re.search(r"sm_(?!100a)\d+", out)


def test_no_cpu_fallback_without_device():
    import torch
    import paper_2503_13092_b200 as pk
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    assert pk.ds_version() == 1 and pk.ds_error_string(pk.ds.DS_E_NOGEOM) == "geometry not uploaded"
    with pytest.raises(pk.DsError) as e:
        pk.ds_create(0)
    assert e.value.code == pk.ds.DS_E_CUDA
    with pytest.raises(RuntimeError):
        import gen
        pk.Downstream(gen.constants.GEOMETRY, gen.mlp_weights(0), gen.constants.PARAMS)


def test_product_never_touches_the_oracle():
    """Neither the package nor the generators import, read or link anything under oracle/ (and vice versa)."""
    for sub in ("paper_2503_13092_b200", "gen"):
        for dp, _, fs in os.walk(os.path.join(ROOT, sub)):
            for f in fs:
                if f.endswith((".py", ".cu", ".cuh", ".h")):
                    txt = open(os.path.join(dp, f)).read()
                    assert not re.search(r"^\s*(from|import)\s+oracle\b|ds_oracle|libds_oracle", txt, flags=re.M), os.path.join(dp, f)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2503_13092_b200" not in txt and "ds.h" not in txt and "libds.so" not in txt
