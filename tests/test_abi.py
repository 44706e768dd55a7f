"""The C-ABI library loads without a GPU and exports every function include/*.h declares (no compute calls)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions(headers=("allen_velo.h", "allen_velo_debug.h", "allen_velo_noalloc.h")):
    names = []
    for h in headers:
        text = open(os.path.join(ROOT, "include", h)).read()
        text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
        names += re.findall(r"\b(allen_velo_[a-z_]+)\s*\(", text)
    return sorted(set(names))


def test_header_declares_the_three_calls_of_the_north_star():
    names = declared_functions(("allen_velo.h",))
    for n in ("allen_velo_create", "allen_velo_reconstruct", "allen_velo_destroy"):
        assert n in names
    # measurement hooks live in their own header, not in the product ABI
    assert not [n for n in names if "timing" in n or "kernel_" in n or "launch_count" in n]
    assert "allen_velo_enable_timing" in declared_functions(("allen_velo_debug.h",))


def test_library_exports_every_declared_symbol():
    from paper_1912_09161_b200 import build

    lib = ctypes.CDLL(build.build())
    for name in declared_functions():
        assert hasattr(lib, name), name


def test_calls_that_need_no_device():
    from paper_1912_09161_b200 import binding

    lib = binding.load_library()
    p = binding.allen_velo_default_params()
    assert (p.w_seed_phi16, p.w_fwd_phi16, p.max_skipped) == (512, 512, 1)
    assert (p.max_slope, p.s_seed, p.s_fwd, p.s_weak) == (ctypes.c_float(0.4).value, 2.0 ** -6, 2.0 ** -4, 2.0 ** -7)
    names = [lib.allen_velo_kernel_name(i).decode() for i in range(lib.allen_velo_kernel_count())]
    assert "velo_cluster" in names and "velo_seed" in names and "velo_follow" in names
    # null handle / null arguments are rejected, not dereferenced
    assert lib.allen_velo_create(None, None) == binding.ERR_INVALID
    assert lib.allen_velo_workspace_bytes(None, 10, 1000) == 0
    assert lib.allen_velo_set_workspace(None, None, 0) == binding.ERR_INVALID
    assert lib.allen_velo_reconstruct(None, None, None, 0, None, None, None) == binding.ERR_INVALID
    lib.allen_velo_destroy(None)
    # the no-allocation entry point checks its arguments before it touches the device
    rc, text = binding.offsets_noalloc(None, 5, None)
    assert rc == binding.ERR_INVALID and "null pointer" in text
    buf = ctypes.create_string_buffer(256)  # (the pointers are never dereferenced: the size is rejected first)
    rc = lib.allen_velo_offsets_noalloc(ctypes.c_void_p(256), binding.NOALLOC_MAX_COUNTS + 1, ctypes.c_void_p(512), None, buf, 256)
    assert rc == binding.ERR_TOO_LARGE and b"exceeds ALLEN_VELO_NOALLOC_MAX_COUNTS = 4194304" in buf.value


def test_binding_structs_match_the_header_layout():
    """ctypes mirrors of the ABI structs: field order and sizes as the C compiler lays them out."""
    from paper_1912_09161_b200 import binding

    assert ctypes.sizeof(binding.allen_velo_params_t) == 28
    assert ctypes.sizeof(binding.allen_velo_geometry_t) == 24 + 3 * 8 + 28 + 4  # padded to 8
    assert ctypes.sizeof(binding.allen_velo_clusters_t) == 8 + 12 * 8
    assert ctypes.sizeof(binding.allen_velo_tracks_t) == 8 + 8 * 8
    assert ctypes.sizeof(binding.allen_velo_vertices_t) == 8 + 2 * 8  # u32 padded to 8, two pointers
    for struct, fields in ((binding.allen_velo_clusters_t, 13), (binding.allen_velo_tracks_t, 10),
                           (binding.allen_velo_vertices_t, 3), (binding.allen_velo_params_t, 7)):
        assert len(struct._fields_) == fields


def test_product_path_refuses_to_run_without_cuda(geometry):
    import pytest
    import torch

    from paper_1912_09161_b200 import binding

    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        binding.AllenVelo(geometry)


def test_the_no_allocation_entry_point_has_no_allocating_call():
    """include/allen_velo_noalloc.h promises it: the translation unit holds a static device array, looks its address up
    with cudaGetSymbolAddress, and calls nothing that allocates."""
    src = open(os.path.join(ROOT, "paper_1912_09161_b200", "csrc_noalloc", "offsets_static.cu")).read()
    code = re.sub(r"//[^\n]*", "", re.sub(r"/\*.*?\*/", "", src, flags=re.S))
    assert re.search(r"static\s+__device__\s+__align__\(256\)\s+unsigned long long\s+g_offsets_state\[", code)
    assert "cudaGetSymbolAddress" in code
    for banned in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "cudaMallocAsync", "malloc(", "new ", "std::vector", "std::string"):
        assert banned not in code, banned
