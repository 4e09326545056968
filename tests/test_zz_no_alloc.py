"""tdde_snorm_noalloc (include/tdde.h): the entry point that allocates nothing -- Re(c^H S c) with the reduction scratch in a file-scope
static __device__ array -- against the existing path (tdde_norm through a handle), on two calls in a row that share the scratch array.
Collected last on purpose (pytest -x: a failure here hides nothing)."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import tdde_inputs  # noqa: E402

pytestmark = pytest.mark.gpu


def _device_inputs(p, torch):
    S = torch.from_numpy(np.ascontiguousarray(p.S_band, dtype=np.complex128)).cuda()
    cls = torch.from_numpy(np.ascontiguousarray(p.cls_of_chan, dtype=np.int32)).cuda()
    return S, cls


def test_snorm_noalloc_matches_tdde_norm_on_two_calls_in_a_row():
    import torch
    from paper_2512_21697_b200 import Tdde, load_library, snorm_noalloc, snorm_noalloc_setup, NOALLOC_MAX_N
    # 257 x 300 = 77 100 elements: 38 blocks, a ragged last block, channel rows that straddle block boundaries, several kappa-classes
    p = tdde_inputs.make_synthetic(n_ang=257, n_r=150, bandwidth=13, n_terms=5, dt=0.01, n_steps=1, rtol=1e-10, seed=21, name="noalloc")
    prop = Tdde(p)                                                  # the existing path (allocates at create)
    S, cls = _device_inputs(p, torch)
    out = torch.full((1,), -7.0, dtype=torch.float64, device="cuda")
    rng = np.random.default_rng(5)
    c1 = p.c0.copy()
    c2 = 3.0 * (rng.standard_normal(p.n) + 1j * rng.standard_normal(p.n))   # a different vector, ~30 000 x the norm: stale partials would show
    snorm_noalloc_setup()
    got, ref = [], []
    for c in (c1, c2):                                              # two calls in a row on the same scratch array
        cd = prop.to_device(c)
        snorm_noalloc(p.n_ang, p.n_rad, p.n_cls, p.w0, S, cls, cd, out)
        torch.cuda.synchronize()
        got.append(float(out.item()))
        ref.append(prop.norm(cd))
    for g, r in zip(got, ref):
        assert abs(g - r) <= 1e-12 * abs(r), (got, ref)             # the apply tolerance of tests/test_gpu_parity.py
    assert abs(ref[0] - 1.0) < 1e-9 and ref[1] > 1e3                # the two calls really had different answers
    # and once more with the first vector: the array carries the second call's partials now
    snorm_noalloc(p.n_ang, p.n_rad, p.n_cls, p.w0, S, cls, prop.to_device(c1), out)
    torch.cuda.synchronize()
    assert abs(float(out.item()) - ref[0]) <= 1e-12 * abs(ref[0])
    # a definition check that involves neither path: dense quadratic form on a few channels
    cc = c2.reshape(p.n_ang, p.n_rad)
    tot = 0.0
    Sb = np.asarray(p.S_band)
    for a in (0, 100, 256):
        k = int(p.cls_of_chan[a])
        for i in range(p.n_rad):
            for d in range(-p.w0, p.w0 + 1):
                if 0 <= i + d < p.n_rad:
                    tot += (np.conj(cc[a, i]) * Sb[k, i, d + p.w0] * cc[a, i + d]).real
    sub = np.zeros_like(cc)
    sub[[0, 100, 256]] = cc[[0, 100, 256]]
    snorm_noalloc(p.n_ang, p.n_rad, p.n_cls, p.w0, S, cls, prop.to_device(sub.reshape(-1)), out)
    torch.cuda.synchronize()
    assert abs(float(out.item()) - tot) <= 1e-12 * abs(tot)
    # sizes beyond the static array are rejected with a text that names the limit; nothing is launched
    lib = load_library()
    out.fill_(-7.0)
    big_ang = NOALLOC_MAX_N // p.n_rad + 1
    rc = snorm_noalloc(big_ang, p.n_rad, p.n_cls, p.w0, S, cls, prop.to_device(c1), out, check=False)
    torch.cuda.synchronize()
    assert rc == -1 and b"TDDE_NOALLOC_MAX_N" in lib.tdde_last_cuda_error()
    assert float(out.item()) == -7.0
    prop.close()


def test_snorm_noalloc_on_a_side_stream_and_largest_bandwidth():
    """w0 = 13 (hydrogen blocks, several classes) on a non-default stream; device memory in use does not change across the calls."""
    import torch
    from paper_2512_21697_b200 import Tdde, snorm_noalloc, snorm_noalloc_setup
    p = tdde_inputs.make_hydrogen(n_r=60, r_max=50.0, kappa_max=3)
    rng = np.random.default_rng(2)
    c = rng.standard_normal(p.n) + 1j * rng.standard_normal(p.n)
    prop = Tdde(p)
    S, cls = _device_inputs(p, torch)
    cd = prop.to_device(c)
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    ref = prop.norm(cd)
    snorm_noalloc_setup()
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        snorm_noalloc(p.n_ang, p.n_rad, p.n_cls, p.w0, S, cls, cd, out, stream=st)      # first launch: module / kernel load happens here
        st.synchronize()
        free0, _ = torch.cuda.mem_get_info()
        for _ in range(2):
            snorm_noalloc(p.n_ang, p.n_rad, p.n_cls, p.w0, S, cls, cd, out, stream=st)
        st.synchronize()
        free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0                                           # nothing was allocated (or freed) by the calls
    assert abs(float(out.item()) - ref) <= 1e-12 * abs(ref)
    prop.close()
