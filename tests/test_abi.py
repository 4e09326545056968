"""CPU-side checks of the boundary: libtdde.so builds, loads and exports every symbol include/tdde.h declares;
the ctypes structs match the header; the product path fails loudly without a GPU (no CPU fallback)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import tdde_inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2512_21697_b200.build import build
    build()
    import paper_2512_21697_b200 as pkg
    return pkg.load_library()


def header_functions(names=("tdde.h", "tdde_bench.h")):
    out = set()
    for name in names:
        src = open(os.path.join(ROOT, "include", name)).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        out |= set(re.findall(r"\b(tdde_[a-z0-9_]+)\s*\(", src))
    return sorted(out)


def test_every_declared_symbol_is_exported(lib):
    import paper_2512_21697_b200 as pkg
    names = header_functions()
    product = set(header_functions(("tdde.h",)))
    assert {"tdde_create", "tdde_step", "tdde_propagate", "tdde_norm", "tdde_apply", "tdde_precond", "tdde_project",
            "tdde_destroy", "tdde_strerror"} <= product
    # measurement helpers, test exports and the comparator are NOT part of the product header
    assert not product & {"tdde_time_kernel", "tdde_fp64_peak", "tdde_selftest_partition", "tdde_paper_variant",
                          "tdde_launch_count", "tdde_step_forced"}
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(pkg.EXPORTS) == names


def test_struct_layouts_match_header():
    import paper_2512_21697_b200 as pkg
    assert C.sizeof(pkg.tdde_config) == 6 * 4 + 2 * 8
    assert C.sizeof(pkg.tdde_term) == 8 + 4 * 8
    assert C.sizeof(pkg.tdde_stats) == 4 * 8 + 8 + 2 * 4
    assert pkg.tdde_config.dt.offset == 24 and pkg.tdde_stats.status.offset == 40


def test_strerror_and_version(lib):
    assert lib.tdde_version() == 2
    assert lib.tdde_strerror(0) == b"ok"
    for code in range(-6, 0):
        assert lib.tdde_strerror(code) not in (b"ok", b"unknown status")
    assert lib.tdde_strerror(-99) == b"unknown status"


def test_create_rejects_bad_arguments_before_touching_cuda(lib):
    import paper_2512_21697_b200 as pkg
    p = tdde_inputs.make_config("tiny")
    h = C.c_void_p()
    S = np.ascontiguousarray(p.S_band)
    H0 = np.ascontiguousarray(p.H0_band)
    cls = np.ascontiguousarray(p.cls_of_chan)

    def cfg(**kw):
        d = dict(n_ang=p.n_ang, n_rad=p.n_rad, n_cls=p.n_cls, w0=p.w0, n_terms=0, max_iter=10, dt=0.01, rtol=1e-10)
        d.update(kw)
        return pkg.tdde_config(d["n_ang"], d["n_rad"], d["n_cls"], d["w0"], d["n_terms"], d["max_iter"], d["dt"], d["rtol"])

    def create(c, cls_arr=cls, S_ptr=None):
        return lib.tdde_create(C.byref(h), C.byref(c), S.ctypes.data if S_ptr is None else S_ptr, H0.ctypes.data,
                               cls_arr.ctypes.data, None, None)

    assert create(cfg(n_ang=0)) == -1
    assert create(cfg(w0=p.n_rad)) == -1
    assert create(cfg(w0=0)) == -1
    assert create(cfg(dt=0.0)) == -1
    assert create(cfg(max_iter=0)) == -1
    assert create(cfg(n_terms=1)) == -1            # terms pointer is NULL
    assert create(cfg(n_terms=99)) == -1
    bad_cls = cls.copy()
    bad_cls[3] = p.n_cls
    assert create(cfg(), cls_arr=bad_cls) == -1
    assert lib.tdde_create(None, C.byref(cfg()), S.ctypes.data, H0.ctypes.data, cls.ctypes.data, None, None) == -1
    assert h.value is None


def test_no_cpu_fallback():
    """Without a CUDA device the product must refuse to run rather than compute on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import paper_2512_21697_b200 as pkg
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        pkg.Tdde(tdde_inputs.make_config("tiny"))
    # and the C ABI itself reports a CUDA error for a valid problem
    lib = pkg.load_library()
    p = tdde_inputs.make_config("tiny")
    c = pkg.tdde_config(p.n_ang, p.n_rad, p.n_cls, p.w0, 0, 10, 0.01, 1e-10)
    h = C.c_void_p()
    S = np.ascontiguousarray(p.S_band); H0 = np.ascontiguousarray(p.H0_band); cls = np.ascontiguousarray(p.cls_of_chan)
    rc = lib.tdde_create(C.byref(h), C.byref(c), S.ctypes.data, H0.ctypes.data, cls.ctypes.data, None, None)
    assert rc == -3 and h.value is None
    assert len(lib.tdde_last_cuda_error()) > 0


def test_product_does_not_import_oracle():
    pkg_dir = os.path.join(ROOT, "paper_2512_21697_b200")
    for dirpath, _, files in os.walk(pkg_dir):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2512_21697_b200" not in txt and "libtdde" not in txt, f


@pytest.mark.parametrize("n,w,P", [(128, 3, 4), (400, 13, 3), (2000, 6, 9), (4000, 6, 74), (97, 3, 16), (64, 9, 1),
                                   (1000, 9, 17), (50, 6, 8), (4000, 9, 60), (400, 13, 6), (200, 1, 10), (31, 2, 3),
                                   (1000, 5, 20), (777, 11, 13)])
def test_partitioned_factorisation_host(lib, n, w, P):
    """Host set-up of the partitioned preconditioner solve (tdde_partition.cu: left spikes W = A_SI A_II^-1, corner blocks,
    block-Thomas factors of the Schur complement) with the three device kernels replayed on the host arrays: the result
    must solve the original banded system to rounding, for ragged sizes, many bandwidths, and plans that shrink."""
    res = C.c_double()
    used = lib.tdde_selftest_partition(n, w, P, 7, C.byref(res))
    assert 1 <= used <= P
    if (n - (P - 1) * w) // P >= max(2 * w, 8):
        assert used == P
    assert res.value < 1e-13, (n, w, P, used, res.value)


@pytest.mark.parametrize("n_rad,w,T", [(8, 3, 1), (37, 3, 7), (64, 6, 5), (101, 6, 7), (50, 9, 7), (19, 9, 2), (7, 6, 3)])
def test_mma_operand_table_host(lib, n_rad, w, T):
    """Host replay of k_apply_mma's radial contraction (tdde_apply_mma.cu: 4-row slices, 8-row tiles, B-operand fragments in lane
    order, complex product by three real ones) against the band product taken from the column bands: radial sizes that are not
    multiples of 8 or 4, sizes smaller than the band, all three instantiated bandwidths; out-of-matrix band entries are poisoned."""
    res = C.c_double()
    assert lib.tdde_selftest_mma_frags(n_rad, w, T, 11, C.byref(res)) == 0
    assert res.value < 1e-13, (n_rad, w, T, res.value)


def test_group_entry_points_reject_bad_arguments(lib):
    """tdde_group_* / tdde_nccl_unique_id (include/tdde.h, NEXT-3): argument errors are reported before any CUDA call."""
    g = C.c_void_p()
    assert lib.tdde_group_create(None, 1, None, None, None) == -1
    assert lib.tdde_group_create(C.byref(g), 0, None, None, None) == -1 and not g.value
    assert lib.tdde_group_create(C.byref(g), 1, None, None, None) == -1 and not g.value
    assert lib.tdde_group_propagate(None, None, 1, None, None) == -1
    assert lib.tdde_nccl_unique_id(None) == -1
    lib.tdde_group_destroy(None)                      # NULL is allowed


def test_reference_arm_prints_on_rank0_only():
    """bench.py --impl reference under a 2-rank launch: rank 0 prints the JSON line, other ranks exit 0 silently."""
    import json
    import subprocess
    import sys
    env = dict(os.environ, WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT="29533")
    outs = []
    for rank in (0, 1):
        r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                            "--warmup", "0", "--config", "tiny", "--sample-ang", "4"], env=dict(env, RANK=str(rank), LOCAL_RANK=str(rank)),
                           capture_output=True, text=True, timeout=600)
        assert r.returncode == 0, r.stderr[-500:]
        outs.append(r.stdout.strip())
    line = json.loads(outs[0].splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0
    assert outs[1] == ""
