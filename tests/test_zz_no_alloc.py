"""tdgl_mean_abs2_static -- the one entry point of libtdgl for callers that cannot allocate device memory.

Who that is: code that sits beside a running solver with nothing but a device pointer to psi -- an in-situ monitor or
logging thread (its cudaMalloc / cudaFree would synchronise the device and stall the time-stepping stream), a plug-in in
an application whose own pool took all of HBM at start-up (cudaMalloc fails there), a component forbidden to allocate
after initialisation.  They have no workspace, hence no tdgl_t handle and no tdgl_observables.  The entry point keeps
the scratch of its reduction (per-CTA partial sums, the counter electing the finishing CTA) in a fixed array inside the
library image instead; the price is a size limit (TDGL_STATIC_MAX_SITES), 64.25 KiB held on every GPU that loads the
library, and one call at a time per device.  include/tdgl.h states the contract.

The GPU tests compare it with the existing path (tdgl_observables -> mean_abs2, whose partial sums live in the caller's
workspace) on two calls in a row: the array is shared by all calls and keeps the previous call's contents, so the second
call is the one that shows a counter or a partial sum left behind by the first.  Tolerance: the 1e-6 absolute that
tests/test_gpu_kernels.py::test_observables uses for <|psi|^2> (both sides add fp32 |psi_m|^2 in fp64, in different orders).

The tests here allocate with torch -- a test may; the entry point under test must not and does not.

This file is named to be collected LAST (pytest --collect-only): `pytest -x` stops at the first failure, and a failure
here must not hide the parity tests.  It passes alone in a fresh process (then its first call does the per-device
set-up) and after the other files (then the library is already loaded and other kernels have run).
"""
import ctypes as C

import numpy as np
import pytest

import tdgl_inputs as I

P_, O_ = I.PERIODIC, I.OPEN
TOL = 1e-6                      # test_observables' tolerance on mean_abs2
CHUNK = 65536                   # sites per partial sum (static_scratch.cu), to place sizes around chunk borders


@pytest.fixture(scope="module")
def B():
    from paper_1409_8340_b200 import build
    build.build()
    from paper_1409_8340_b200 import binding
    binding.lib()
    return binding


# ---- host-side contract: every rejection happens before the first CUDA call, so these run without a GPU ---------------
def test_rejects_what_the_builtin_scratch_cannot_cover(B):
    L = B.lib()
    fake_psi, fake_out = C.c_void_p(0x1000), C.c_void_p(0x2000)       # never dereferenced: the call must return first
    assert B.TDGL_STATIC_MAX_SITES == 1024 * 1024 * 512
    assert L.tdgl_mean_abs2_static(fake_psi, B.TDGL_STATIC_MAX_SITES + 1, fake_out, None) == B.TDGL_ESCRATCH
    assert L.tdgl_mean_abs2_static(fake_psi, 1 << 40, fake_out, None) == B.TDGL_ESCRATCH
    assert "TDGL_STATIC_MAX_SITES" in B.tdgl_strerror(B.TDGL_ESCRATCH)
    with pytest.raises(B.TdglError) as e:
        B.tdgl_mean_abs2_static(0x1000, B.TDGL_STATIC_MAX_SITES + 1, 0x2000)
    assert e.value.code == B.TDGL_ESCRATCH
    for psi, n, out in ((None, 16, fake_out), (fake_psi, 16, None), (fake_psi, 0, fake_out), (fake_psi, -3, fake_out),
                        (C.c_void_p(0x1004), 16, fake_out), (fake_psi, 16, C.c_void_p(0x2004))):
        assert L.tdgl_mean_abs2_static(psi, n, out, None) == B.TDGL_EINVAL


def test_header_states_the_limit_and_the_sharing_rule():
    import os
    src = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "tdgl.h")).read()
    assert "#define TDGL_STATIC_MAX_SITES     536870912" in src and "#define TDGL_STATIC_SCRATCH_BYTES 65792" in src
    doc = src[src.index("for callers that cannot allocate device memory"):src.index("int tdgl_mean_abs2_static")]
    for word in ("cudaGetSymbolAddress", "before any stream capture", "race", "TDGL_ESCRATCH", "until the process exits"):
        assert word in doc, word


# ---- GPU ----------------------------------------------------------------------------------------------------------------
def _static_mean(B, torch, psi_c64, out=None, slot=0):
    """One call of the entry point on torch's current stream; `psi_c64` is a contiguous complex64 device tensor."""
    if out is None:
        out = torch.full((4,), float("nan"), dtype=torch.float64, device=psi_c64.device)
    B.tdgl_mean_abs2_static(psi_c64.data_ptr(), psi_c64.numel(), out.data_ptr() + 8 * slot,
                            torch.cuda.current_stream(psi_c64.device).cuda_stream)
    return out


@pytest.mark.gpu
def test_two_calls_in_a_row_agree_with_tdgl_observables(B):
    torch = pytest.importorskip("torch")
    from gpu_common import setup_pair
    # 4.5 chunks: several CTAs and a ragged last one; pinning, field and current so that |psi|^2 varies and evolves
    cfg = I.Config("na", 128, 96, 24, (P_, P_, O_), nz_flux=6, Jx=0.02, incl_fraction=0.15, incl_rmin=1.0, incl_rmax=2.0)
    rng = np.random.default_rng(11)
    shape = (cfg.nz, cfg.ny, cfg.nx)
    psi0 = ((0.6 + 0.4 * rng.uniform(-1, 1, shape)) * np.exp(1j * rng.uniform(-np.pi, np.pi, shape))).astype(np.complex64)
    _, _, _, _, s = setup_pair(cfg, psi0=psi0)
    out = torch.full((4,), float("nan"), dtype=torch.float64, device="cuda")
    seen = []
    for call in range(2):                                   # two calls in a row on DIFFERENT states: the first leaves the
        s.step(4)                                           # shared array dirty (8192-entry partial sums, counter = 5)
        psi, _ = s.get_psi_mu()
        ref = s.observables().mean_abs2                     # existing path: partial sums in the caller's workspace
        _static_mean(B, torch, psi, out, slot=call)
        torch.cuda.synchronize()
        got = float(out[call])
        host = float(np.mean(np.abs(psi.cpu().numpy().astype(np.complex128)) ** 2))
        assert abs(got - ref) < TOL, (call, got, ref)
        assert abs(got - host) < TOL, (call, got, host)
        seen.append(got)
    assert abs(seen[0] - seen[1]) > 1e-5                    # the state did move: the second call did not echo the first
    assert torch.isnan(out[2:]).all()                       # one double written per call, nothing beyond it
    # and back to back with no host work in between, same input: the fixed summation order gives the same bits
    a = torch.full((4,), float("nan"), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]              # device-wide: would also see a cudaMalloc made by the library
    _static_mean(B, torch, psi, a, slot=0)
    _static_mean(B, torch, psi, a, slot=1)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before      # set-up happened in the first call above; these took nothing
    assert float(a[0]) == float(a[1]) == seen[1]
    s.close()


@pytest.mark.gpu
@pytest.mark.parametrize("n,offset", [(1, 0), (2, 0), (3, 1), (CHUNK - 1, 0), (CHUNK, 1), (CHUNK + 1, 0), (5 * CHUNK + 777, 1),
                                      (7 * CHUNK, 0)])
def test_sizes_around_chunk_borders_and_unaligned_views(B, n, offset):
    """A large call first, then the small one: a shorter grid must not pick up partial sums or the counter the longer one
    left in the shared array.  offset = 1 site makes psi 8-byte but not 16-byte aligned (the one-site-per-load path)."""
    torch = pytest.importorskip("torch")
    g = torch.Generator(device="cuda").manual_seed(1000 + n)
    big = torch.randn(9 * CHUNK + 5, 2, generator=g, device="cuda", dtype=torch.float32)
    small = torch.view_as_complex(torch.randn(n + offset, 2, generator=g, device="cuda", dtype=torch.float32))[offset:]
    assert small.data_ptr() % 16 == (8 if offset else 0)
    out = _static_mean(B, torch, torch.view_as_complex(big), slot=0)
    _static_mean(B, torch, small, out, slot=1)
    torch.cuda.synchronize()
    for slot, t in ((0, torch.view_as_complex(big)), (1, small)):
        ref = float((torch.view_as_real(t).double() ** 2).sum() / t.numel())
        assert abs(float(out[slot]) - ref) < TOL * max(1.0, ref), (slot, float(out[slot]), ref)


@pytest.mark.gpu
def test_headline_mesh_and_the_maximum_size(B):
    """C4 (512 x 512 x 256) and exactly TDGL_STATIC_MAX_SITES = C5 (1024 x 1024 x 512, 4 GiB of psi): every one of the
    8192 partial sums is in use at the maximum."""
    torch = pytest.importorskip("torch")
    free, _ = torch.cuda.mem_get_info()
    for n in (512 * 512 * 256, B.TDGL_STATIC_MAX_SITES):
        if free < 10 * n:                                   # psi itself is 8 B/site; the reference below works in slices
            pytest.skip("not enough free device memory for the reference")
        x = torch.empty(n, 2, device="cuda", dtype=torch.float32)
        g = torch.Generator(device="cuda").manual_seed(n % 1000)
        step = 1 << 24
        ref = 0.0
        for lo in range(0, n, step):                        # fill and reference in slices of 16 M sites
            x[lo:lo + step].uniform_(-1.0, 1.0, generator=g)
            ref += float((x[lo:lo + step].double() ** 2).sum())
        ref /= n
        out = _static_mean(B, torch, torch.view_as_complex(x))
        torch.cuda.synchronize()
        assert abs(float(out[0]) - ref) < TOL, (n, float(out[0]), ref)
        assert abs(ref - 2.0 / 3.0) < 1e-3                  # E|psi|^2 of two uniform(-1, 1) components
        del x
