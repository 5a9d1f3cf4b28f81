"""cav_diag_noalloc: the a4 diagnostics for callers that may not allocate device memory.

Who needs it: code that runs while a stream of the process is being captured in the global capture mode (cudaMalloc is
refused there and spoils the capture), a solver confined to a slice of HBM somebody else handed it (the rest of the GPU is
another framework's pool), and loops that cannot take the device-wide synchronisation of cudaMalloc / cudaFree.  They keep
psi and omega in device buffers of their own, so they can use neither cav_create (which takes its fields from PyTorch's
caching allocator) nor cav_get_diag (which needs a context).  The entry point takes their device pointers and keeps its
partial sums in a fixed array inside the library image; that array is why N is limited to CAV_NOALLOC_MAX_N = 8192, why
it is shared by all calls (so calls that overlap on the GPU would race), and why stale contents of an earlier call are
the thing to test for.

The GPU tests compare it with the existing path (cav_create -> cav_set_fields -> cav_get_diag) within the 1e-9 relative
tolerance the other diagnostics tests use (the sums are folded in a different order, so not bit for bit), on calls made
back to back on one stream: a large grid, then a small one (whose fold must not see the large grid's leftover slots), then
the large one again (which must repeat its first answer bit for bit).

This file is named so that pytest collects it last: with `pytest -x` a failure here hides nothing else.
"""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
KEYS = ("res_inf", "res_l2", "kinetic_energy", "enstrophy")
TOL = 1e-9        # as tests/test_gpu_parity.py uses for the a4 sums


@pytest.fixture(scope="module")
def cav():
    from paper_0809_3098_b200 import binding
    binding.lib()
    return binding


def state(N, seed):
    """A seeded (psi, omega) pair with psi = 0 on the walls, as cav_set_fields would leave it."""
    rng = np.random.default_rng(seed)
    psi = 0.05 * rng.standard_normal((N + 1, N + 1))
    psi[0, :] = psi[N, :] = 0.0
    psi[:, 0] = psi[:, N] = 0.0
    w = 3.0 * rng.standard_normal((N + 1, N + 1))
    return psi, w


def existing_path(cav, N, psi, w):
    """cav_create -> cav_set_fields -> cav_get_diag: the allocating path the new entry point is measured against."""
    with cav.Cavity(N, 100.0, 1e-3, 1.5, 1) as c:
        c.set_fields(psi, w)
        d = c.diag()
    return np.array([d[k] for k in KEYS])


def to_device(a, pitch):
    """Host (N+1, N+1) array -> CUDA tensor of (N+1) rows of `pitch` doubles; the padding holds NaN (it must never be read)."""
    import torch
    t = torch.full((a.shape[0], pitch), float("nan"), dtype=torch.float64, device="cuda")
    t[:, : a.shape[1]] = torch.from_numpy(a).cuda()
    return t


def close(a, b):
    return np.all(np.abs(a - b) <= TOL * np.abs(b))


@pytest.mark.gpu
def test_noalloc_matches_get_diag_on_calls_in_a_row(cav):
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    torch.cuda.set_device(0)
    # (N, pitch): large dense; small dense right after it (leftover slots 63.. of the first call); the large one again;
    # padded rows; the smallest grid there is (one interior point, one CTA)
    cases = [(257, 258), (64, 65), (257, 258), (1000, 1004), (2, 3)]
    states = {N: state(N, 1000 + N) for N, _ in cases}
    want = {N: existing_path(cav, N, *states[N]) for N in states}
    dev = {(N, p): (to_device(states[N][0], p), to_device(states[N][1], p)) for N, p in set(cases)}
    outs = [torch.full((4,), float("nan"), dtype=torch.float64, device="cuda") for _ in cases]
    st = torch.cuda.current_stream().cuda_stream
    for (N, p), out in zip(cases, outs):              # back to back on one stream, no host synchronisation in between
        psi_d, w_d = dev[(N, p)]
        cav.diag_noalloc(N, psi_d, w_d, out, pitch=p, stream=st)
    torch.cuda.synchronize()
    got = [o.cpu().numpy() for o in outs]
    for (N, p), g in zip(cases, got):
        assert np.all(np.isfinite(g)), (N, g)
        assert close(g, want[N]), (N, p, g, want[N])
        assert g[0] == want[N][0], "res_inf is a maximum: no rounding to differ by"
    assert np.array_equal(got[0], got[2]), "same input, same answer bit for bit, whatever ran in between"
    # and against the CPU oracle's a4 (the definitions of struct cav_diag written out in plain loops), same tolerance
    import oracle
    for N in (64, 257):
        o = oracle.OracleCavity(N, 100.0, 1e-3, 1.5, 1)
        o.set_fields(*states[N])
        od = o.diag()
        o.close()
        g = got[[c[0] for c in cases].index(N)]
        assert close(g, np.array([od[k] for k in KEYS])), (N, g, od)


@pytest.mark.gpu
def test_noalloc_on_a_side_stream_and_at_the_limit(cav):
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    torch.cuda.set_device(0)
    N = cav.noalloc_max_n()                           # 8192: every slot of the fixed scratch in use
    assert N == 8192
    rng = np.random.default_rng(8192)
    psi = rng.standard_normal((N + 1, N + 1)) * 0.05
    psi[0, :] = psi[N, :] = 0.0
    psi[:, 0] = psi[:, N] = 0.0
    w = rng.standard_normal((N + 1, N + 1)) * 3.0
    want = existing_path(cav, N, psi, w)
    psi_d, w_d = torch.from_numpy(psi).cuda(), torch.from_numpy(w).cuda()
    out = torch.zeros(4, dtype=torch.float64, device="cuda")
    out2 = torch.zeros(4, dtype=torch.float64, device="cuda")
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        cav.diag_noalloc(N, psi_d, w_d, out, stream=side.cuda_stream)
        cav.diag_noalloc(N, psi_d, w_d, out2, stream=side.cuda_stream)
    side.synchronize()
    g, g2 = out.cpu().numpy(), out2.cpu().numpy()
    assert close(g, want), (g, want)
    assert np.array_equal(g, g2)


def test_noalloc_rejects_what_does_not_fit(cav):
    """Argument checks come before any CUDA call, so they can be tested without a GPU; nothing is dereferenced."""
    L = cav.lib()
    p = C.c_void_p(4096)                              # any non-null address: a rejected call must not touch it
    nmax = L.cav_noalloc_max_n()
    assert nmax == 8192
    assert L.cav_diag_noalloc(nmax + 1, nmax + 2, p, p, p, None) == -5          # CAV_ELIMIT
    assert b"CAV_NOALLOC_MAX_N" in L.cav_strerror(-5)
    with pytest.raises(cav.CavityError, match="CAV_NOALLOC_MAX_N"):
        cav.diag_noalloc(nmax + 1, p.value, p.value, p.value)
    assert L.cav_diag_noalloc(1, 2, p, p, p, None) == -1                        # CAV_EINVAL: N < 2
    assert L.cav_diag_noalloc(64, 64, p, p, p, None) == -1                      # pitch < N + 1
    assert L.cav_diag_noalloc(64, 65, None, p, p, None) == -1
    assert L.cav_diag_noalloc(64, 65, p, None, p, None) == -1
    assert L.cav_diag_noalloc(64, 65, p, p, None, None) == -1


def test_noalloc_source_calls_no_allocator():
    """The promise of the entry point, checked on its source: no allocating call anywhere in the file (comments aside),
    the scratch is a file-scope static __device__ array, and its address comes from cudaGetSymbolAddress."""
    src = open(os.path.join(ROOT, "paper_0809_3098_b200", "csrc", "cavity_noalloc.cu")).read()
    code = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    code = re.sub(r"//[^\n]*", "", code)
    for banned in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "raw_alloc", "CachingAllocator", "cudaMemPool", "new ", "malloc("):
        assert banned not in code, banned
    assert re.search(r"static\s+__device__\s+__align__\(256\)", code)
    assert "cudaGetSymbolAddress" in code
