"""cbct_quality_metrics_static: the entry point that allocates nothing (its scratch is a file-scope static __device__ array in
metrics_static.cu).  Collected last on purpose (the suite runs with pytest -x): a failure here hides no other test.

The existing path (cbct_quality_metrics, scratch allocated by cbct_geometry_create) is the reference: same six fp64 sums in
another fixed order, so e and c agree to fp64 rounding; the tolerance is the one tests/test_metrics.py uses (rel 1e-10).
Two calls in a row on different inputs: the second must not see anything the first left in the shared scratch."""
import numpy as np
import pytest

from paper_1001_0599_b200 import inputs as I

TOL = 1e-10


def _volumes(shape, seed):
    nz, ny, nx = shape
    g = I.Geometry(nx=nx, ny=ny, nz=nz, hx=1.0, hy=1.0, hz=1.0, nu=16, nv=16, du=4.0, dv=4.0, n_proj=2)
    f0 = I.uniform_volume(g, seed)
    f = (f0 * 0.9 + 0.002 * I.uniform_volume(g, seed + 1, hi=1.0)).astype(np.float32)
    return g, f, f0


@pytest.mark.gpu
def test_static_metrics_match_the_handle_path_on_two_calls_in_a_row():
    import torch
    from paper_1001_0599_b200 import cbct
    # several blocks with a ragged last chunk (19 * 45 * 37 = 31 635 = 1 chunk + 15 251), then 16 whole chunks
    cases = [((19, 45, 37), 81), ((64, 64, 64), 91)]
    want, devs = [], []
    for shape, seed in cases:
        g, f, f0 = _volumes(shape, seed)
        a, b = torch.from_numpy(f).cuda(), torch.from_numpy(f0).cuda()
        with cbct.geometry_create(g) as h:
            want.append(h.quality_metrics(a, b))
        devs.append((a, b))
    # the two calls back to back on one stream, each into its own output; read only after both were issued
    outs = [torch.full((2,), -7.0, device="cuda", dtype=torch.float64) for _ in cases]
    for (a, b), o in zip(devs, outs):
        cbct.quality_metrics_static(a, b, o)
    torch.cuda.synchronize()
    for (we, wc), o in zip(want, outs):
        e, c = o.cpu().tolist()
        assert e == pytest.approx(we, rel=TOL) and c == pytest.approx(wc, rel=TOL), (e, we, c, wc)
    # the same call again gives the same bits (fixed summation order, nothing left over in the scratch) ...
    again = torch.zeros(2, device="cuda", dtype=torch.float64)
    cbct.quality_metrics_static(devs[0][0], devs[0][1], again)
    torch.cuda.synchronize()
    assert again.cpu().numpy().tobytes() == outs[0].cpu().numpy().tobytes()
    # ... a volume against itself is (0, 1), a prefix of a buffer is honoured (n < numel)
    same = torch.zeros(2, device="cuda", dtype=torch.float64)
    cbct.quality_metrics_static(devs[1][1], devs[1][1], same)
    part = torch.zeros(2, device="cuda", dtype=torch.float64)
    n = 20000
    cbct.quality_metrics_static(devs[1][0], devs[1][1], part, n=n)
    torch.cuda.synchronize()
    assert same.cpu().tolist() == [0.0, pytest.approx(1.0, abs=1e-12)]
    fa, fb = devs[1][0].cpu().numpy().ravel()[:n].astype(np.float64), devs[1][1].cpu().numpy().ravel()[:n].astype(np.float64)
    assert part[0].item() == pytest.approx(np.linalg.norm(fa - fb) / np.linalg.norm(fb), rel=TOL)
    assert part[1].item() == pytest.approx(np.corrcoef(fa, fb)[0, 1], rel=TOL)


@pytest.mark.gpu
def test_static_metrics_refuse_sizes_beyond_the_scratch():
    import torch
    from paper_1001_0599_b200 import cbct
    a = torch.zeros(8, device="cuda", dtype=torch.float32)
    out = torch.full((2,), 5.0, device="cuda", dtype=torch.float64)
    with pytest.raises(cbct.CbctError) as ei:
        cbct.quality_metrics_static(a, a, out, n=cbct.STATIC_MAX_ELEMS + 1)      # refused before anything is read
    assert "exceeds the static scratch's maximum" in str(ei.value)
    with pytest.raises(cbct.CbctError):
        cbct.quality_metrics_static(a, a, out, n=0)
    torch.cuda.synchronize()
    assert out.cpu().tolist() == [5.0, 5.0]                                       # nothing was launched
    cbct.quality_metrics_static(a, a, out)                                        # and the entry point still works: all-zero volumes
    torch.cuda.synchronize()
    assert out.cpu().tolist() == [0.0, 0.0]


def test_static_metrics_argument_checks_need_no_gpu():
    """NULL buffers, n = 0 and n beyond CBCT_STATIC_MAX_ELEMS are refused before the first CUDA call: checked here without a
    device (the pointers are never dereferenced)."""
    import ctypes as C
    from paper_1001_0599_b200 import cbct
    lib = cbct.load_library()
    fake = C.c_void_p(0x1000)
    call = lib.cbct_quality_metrics_static
    assert call(None, fake, C.c_ulonglong(8), fake, None) == 1                     # CBCT_ERR_INVALID_ARG
    assert call(fake, fake, C.c_ulonglong(8), None, None) == 1
    assert call(fake, fake, C.c_ulonglong(0), fake, None) == 1
    assert call(fake, fake, C.c_ulonglong(cbct.STATIC_MAX_ELEMS + 1), fake, None) == 1
    assert b"CBCT_STATIC_MAX_ELEMS" in lib.cbct_last_error()
    # the header's limits are the binding's
    import os, re
    text = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "cbct.h")).read()
    assert int(re.search(r"#define CBCT_STATIC_MAX_ELEMS (\d+)ull", text).group(1)) == cbct.STATIC_MAX_ELEMS
    chunk = int(re.search(r"#define CBCT_STATIC_CHUNK (\d+)", text).group(1))
    blocks = int(re.search(r"#define CBCT_STATIC_MAX_BLOCKS (\d+)", text).group(1))
    assert chunk * blocks == cbct.STATIC_MAX_ELEMS
