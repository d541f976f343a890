"""C-ABI checks that need no GPU: the library loads, exports every symbol include/set.h declares, the ctypes
structs agree with the C structs, and calls fail cleanly (no abort, no CPU fallback) without a device."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "set.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(set_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(libset):
    lib = libset.load()
    declared = _declared_symbols()
    assert len(declared) >= 19
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in include/set.h but not exported by libset.so"
    assert sorted(libset.EXPORTS) == declared


def test_builtin_descriptors_roundtrip_struct_layout(libset):
    # if the ctypes mirrors of set_stage_desc / set_buffer_desc were laid out differently from the C structs
    # these fields would come back as garbage
    st, ns, bf, nb, hin, hout = libset.builtin_pipeline(0)
    assert (ns, nb, hin, hout) == (2, 2, 16384, 16640)
    assert st[0].block[0] == 1024 and st[1].block[0] == 256 and st[0].num_args == 3 and st[0].args[2].kind == libset.ARG_IMM32 and st[0].args[2].imm == 4096
    assert st[1].args[1].kind == libset.ARG_BUFFER and st[1].args[1].index == 1 and st[1].args[1].offset.fixed == 16384
    assert bf[0].h2d_bytes.fixed == 16384 and bf[1].d2h_bytes.fixed == 16640 and bf[1].bytes == 16640
    assert st[0].func == libset.load().set_builtin_kernel(1) and st[0].func
    st, ns, bf, nb, hin, hout = libset.builtin_pipeline(1)
    assert (ns, nb, hin, hout) == (5, 3, 131072, 4) and st[0].grid[0].count.fixed == 16
    st, ns, bf, nb, hin, hout = libset.builtin_pipeline(2)
    assert (ns, nb, hin, hout) == (10, 2, 4096 * 4096 * 4, 4096 * 4096 * 4) and bf[0].d2h_bytes.fixed == hout
    st, ns, bf, nb, hin, hout = libset.builtin_pipeline(2, params=[64, 64, 3])
    assert ns == 3 and bf[1].d2h_bytes.fixed == 64 * 64 * 4 and bf[0].d2h_bytes.fixed == 0      # odd sweep count ends in buffer 1
    st, ns, bf, nb, hin, hout = libset.builtin_pipeline(3)
    assert (ns, nb, hin, hout) == (1, 2, 16785408, 8388608) and st[0].args[0].kind == libset.ARG_TMAP2D
    assert st[0].args[1].offset.fixed == 8388608 and st[0].args[1].tmap.inner == 2048 and st[0].smem_bytes > 48 * 1024
    st, ns, bf, nb, hin, hout = libset.builtin_pipeline(4)
    assert (ns, nb, hin, hout) == (3, 4, 6220800, 2073600 + 1024)
    assert bf[0].h2d_bytes.per_unit == 3 and bf[0].h2d_bytes.dim_mask == 3 and bf[3].flags == libset.BUF_ZERO
    assert bf[3].d2h_host_off.per_unit == 1 and st[1].block[0] == 32 and st[1].block[1] == 4
    st, ns, bf, nb, _, _ = libset.builtin_pipeline(0, variant=libset.VARIANT_SPIN)
    assert ns == 3 and nb == 3 and st[2].args[1].kind == libset.ARG_DIM and st[2].args[1].index == 3
    with pytest.raises(libset.SetError):
        libset.builtin_pipeline(7)
    # degenerate sizes are rejected when the descriptors are built (an empty job has no graph)
    for config, params in ((0, [0]), (1, [0]), (2, [0, 16, 1]), (2, [16, 16, 0]), (2, [16, 16, 17]), (3, [0, 8, 8]), (3, [8, 12, 8]), (4, [0, 4])):
        with pytest.raises(libset.SetError):
            libset.builtin_pipeline(config, params=params)
    assert libset.load().set_builtin_kernel(99) is None


def test_every_builtin_kernel_id_in_the_header_resolves(libset):
    text = open(os.path.join(ROOT, "include", "set.h")).read()
    ids = {name: int(v) for name, v in re.findall(r"#define\s+(SET_K_[A-Z0-9_]+)\s+(\d+)", text)}
    assert len(ids) >= 15 and sorted(ids.values()) == list(range(1, len(ids) + 1))
    lib = libset.load()
    for name, v in ids.items():
        assert lib.set_builtin_kernel(v), f"{name} = {v} has no entry in set_builtin_kernel()"


def test_struct_sizes_match_header(libset):
    assert C.sizeof(libset.SizeExpr) == 24 and C.sizeof(libset.GridRule) == 32 and C.sizeof(libset.Tmap2D) == 40
    assert C.sizeof(libset.ArgDesc) == 8 + 24 + 8 + 40
    assert C.sizeof(libset.Stats) == 20 * 8
    assert C.sizeof(libset.Config) == 14 * 4 + 8 + 8 + 8 + 16
    assert C.sizeof(libset.GapStats) == 13 * 8


def test_invalid_arguments_are_rejected_without_a_device(libset):
    lib = libset.load()
    h = C.c_void_p(None)
    assert lib.set_create(0, 8, C.byref(h)) == libset.SET_ERR_INVALID and not h
    assert lib.set_create(4, 0, C.byref(h)) == libset.SET_ERR_INVALID
    assert lib.set_create(4, 8, None) == libset.SET_ERR_INVALID
    assert lib.set_submit(None, 0, None, None) == libset.SET_ERR_INVALID
    assert lib.set_drain(None) == libset.SET_ERR_INVALID
    assert lib.set_destroy(None) == libset.SET_OK
    assert lib.set_last_error(None) == b""
    assert lib.set_try_submit_dims(None, 0, None, None, None) == libset.SET_ERR_INVALID
    m = C.c_void_p(None)
    assert lib.set_multi_create(None, 2, None, C.byref(m)) == libset.SET_ERR_INVALID and not m
    assert lib.set_multi_submit_dims(None, 0, None, None, None) == libset.SET_ERR_INVALID
    assert lib.set_multi_drain(None) == libset.SET_ERR_INVALID
    assert lib.set_multi_destroy(None) == libset.SET_OK and lib.set_multi_stolen(None) == 0 and not lib.set_multi_instance(None, 0)


def test_no_cpu_fallback_without_gpu(libset):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    lib = libset.load()
    h = C.c_void_p(None)
    assert lib.set_create(4, 8, C.byref(h)) == libset.SET_ERR_CUDA      # fails loudly, does not fall back
    assert not h
    with pytest.raises(libset.SetError):
        libset.Context(4, 8)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2606_05495_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cpp", ".cu", ".hpp", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), f
                assert "oracle.h" not in src and "liboracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2606_05495_b200" not in src.replace("imports nothing from\npaper_2606_05495_b200", "") or f in ("__init__.py", "oracle.h")
            assert not re.search(r"^\s*(import|from)\s+paper_2606_05495_b200", src, flags=re.M), f
            assert "set.h" not in src and "libset" not in src, f


def test_no_global_memory_access_is_scheduled_before_griddepcontrol_wait(libset):
    """Every built-in kernel starts with griddepcontrol.launch_dependents / .wait (kernels.h set_pdl_sync) so that it may sit
    behind a programmatic edge.  The compiler once moved an invariant load (`const T* __restrict__` parameter, ld.global.nc)
    in front of the wait -- a stale read of the slot's previous job -- so the SASS of every kernel is scanned:
    no global load, store, atomic or TMA load may precede ACQBULK (the wait)."""
    import shutil
    import subprocess
    from paper_2606_05495_b200 import build as b
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    objs = [os.path.join(b.BUILD_DIR, f) for f in sorted(os.listdir(b.BUILD_DIR)) if f.startswith("kernels_") and f.endswith(".o")]
    assert len(objs) >= 4
    seen, bad = set(), []
    mem = re.compile(r"\b(LDG|LD\.E|STG|ST\.E|ATOMG?|RED|UTMALDG|UTMASTG)\b")
    for o in objs:
        sass = subprocess.run([cuobjdump, "-sass", o], capture_output=True, text=True, check=True).stdout
        fn, waited = None, False
        for ln in sass.splitlines():
            m = re.search(r"Function : (\S+)", ln)
            if m:
                fn, waited = m.group(1), False
                continue
            if fn is None or not re.search(r"/\*[0-9a-f]{4,}\*/", ln):
                continue
            if "ACQBULK" in ln:
                waited = True
                seen.add(fn)
            elif not waited and mem.search(ln):
                bad.append((fn, ln.strip()[:90]))
    assert not bad, bad[:5]
    kernels = {n for n in seen if n.startswith("set_k_")}
    assert len(kernels) >= 25, sorted(kernels)          # every set_k_* kernel has the wait
