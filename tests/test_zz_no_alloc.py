"""sc_residual_norm_static — the entry point that allocates nothing (include/sc_riccati.h) — against the existing path.

The existing path is the residual of Eq. 27 that sc_iterate reports as stats.res_delta (two-stage reduction
with its partial sums in the context's cudaMalloc'ed scratch).  With the Picard update and step 1 (E5 :1070) the
iterate moves by exactly x_new - x_old = Delta_out - Delta_in, so the static-scratch entry point applied to the order
parameter before and after an iteration must reproduce res_delta, in each of the three norms.  Collected last on
purpose (the suite runs with pytest -x); it depends on no state left by other tests, nor do they on it.
"""
import ctypes as C

import numpy as np
import pytest

import workloads as wlmod

torch = pytest.importorskip("torch")

TOL = 1e-9          # the FP64 tolerance of tests/test_gpu_parity.py


@pytest.fixture(scope="module")
def sc():
    import paper_2205_15000_b200 as m
    from paper_2205_15000_b200 import build
    build.build()
    return m


def test_rejects_sizes_beyond_the_static_scratch_before_touching_the_device(sc):
    """argument checks come first: no GPU needed, nothing is enqueued"""
    L = sc.load_library()
    buf = (C.c_double * 8)()
    err = C.create_string_buffer(256)
    p = C.cast(buf, C.c_void_p)
    rc = L.sc_residual_norm_static(p, p, sc.RESIDUAL_STATIC_MAX_ELEMENTS + 1, 2, p, -1, None, err, len(err))
    assert rc == 1 and b"8388609 elements exceed the static scratch's maximum of 8388608" in err.value
    assert L.sc_residual_norm_static(p, p, 0, 2, p, -1, None, err, len(err)) == 1 and b"n < 1" in err.value
    assert L.sc_residual_norm_static(p, p, 4, 3, p, -1, None, err, len(err)) == 1 and b"norm_p" in err.value
    assert L.sc_residual_norm_static(None, p, 4, 2, p, -1, None, None, 0) == 1
    src = open(sc.lib_path().replace("libsc_riccati.so", "csrc/sc_static.cu")).read().split("#include", 1)[1]
    assert "cudaMalloc" not in src and "cudaFree" not in src and "cudaGetSymbolAddress" in src


@pytest.mark.gpu
@pytest.mark.parametrize("norm_p", [2, 1, -1])
def test_static_scratch_residual_matches_sc_iterate_on_two_calls_in_a_row(sc, norm_p):
    wl = wlmod.make_workload(0)
    ctx = sc.ScContext.from_workload(wl, residual_norm=norm_p)
    d = torch.as_tensor(np.ascontiguousarray(wl.delta0.astype(np.complex128)), device="cuda").clone()
    out = torch.full((3,), float("nan"), dtype=torch.float64, device="cuda")       # allocated by the caller, before the calls
    before = torch.empty_like(d)
    seen = []
    for it in range(2):                                                             # two calls in a row, on different data
        before.copy_(d)
        st = ctx.sc_iterate(0, 1.0, False, d, want_stats=True)                      # Picard, step 1: Delta_out = Delta_in + (g(x) - x)
        torch.cuda.synchronize()
        free = torch.cuda.mem_get_info()[0]                                         # the driver's count: sees a cudaMalloc by the library too
        sc.sc_residual_norm_static(d, before, out, norm_p=norm_p)
        torch.cuda.synchronize()
        if it == 1:                                                                 # (the first call on a device may load the kernels' module)
            assert torch.cuda.mem_get_info()[0] == free
        num, den, ratio = out.cpu().numpy()
        assert st.res_delta > 1e-4                                                  # a real step, not 0 = 0
        assert abs(ratio - st.res_delta) < TOL * st.res_delta, (it, ratio, st.res_delta)
        # and the two norms themselves against the textbook definition
        diff = (d - before).abs().double().flatten(); old = before.abs().double().flatten()
        ref = {2: lambda v: float(torch.linalg.vector_norm(v, 2)), 1: lambda v: float(v.sum()), -1: lambda v: float(v.max())}[norm_p]
        assert abs(num - ref(diff)) < TOL * ref(diff) and abs(den - ref(old)) < TOL * ref(old)
        assert abs(ratio - num / den) <= 1e-15 * ratio
        seen.append(ratio)
    assert seen[0] != seen[1]
    # the same input again: the array keeps the last call's contents, the result must not
    sc.sc_residual_norm_static(d, before, out, norm_p=norm_p)
    assert float(out[2]) == seen[1]
    ctx.close()


@pytest.mark.gpu
def test_static_scratch_at_its_maximum_size_then_a_small_call(sc):
    """All 4096 tiles of the scratch, then 3 tiles and a ragged tail: the partial sums the big call left behind must not leak"""
    g = torch.Generator(device="cuda").manual_seed(5)
    n = sc.RESIDUAL_STATIC_MAX_ELEMENTS
    a = torch.view_as_complex(torch.randn((n, 2), dtype=torch.float64, device="cuda", generator=g))
    b = torch.view_as_complex(torch.randn((n, 2), dtype=torch.float64, device="cuda", generator=g))
    out = torch.zeros(3, dtype=torch.float64, device="cuda")
    for m in (n, 3 * 2048 + 77, 1):
        x, y = a[:m].contiguous(), b[:m].contiguous()
        for p, ref in ((2, lambda v: torch.linalg.vector_norm(v, 2)), (1, torch.sum), (-1, torch.max)):
            sc.sc_residual_norm_static(x, y, out, norm_p=p)
            want = float(ref((x - y).abs())) / float(ref(y.abs()))
            assert abs(float(out[2]) - want) < 1e-12 * want, (m, p)
    with pytest.raises(sc.ScError, match="exceed the static scratch's maximum"):
        big = torch.zeros(n + 1, dtype=torch.complex128, device="cuda")
        sc.sc_residual_norm_static(big, big, out)
    # a side stream: the work is enqueued where the caller says
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        sc.sc_residual_norm_static(a[:5000].contiguous(), b[:5000].contiguous(), out, norm_p=2, stream=s.cuda_stream)
    s.synchronize()
    want = float(torch.linalg.vector_norm((a[:5000] - b[:5000]).abs(), 2) / torch.linalg.vector_norm(b[:5000].abs(), 2))
    assert abs(float(out[2]) - want) < 1e-12 * want
