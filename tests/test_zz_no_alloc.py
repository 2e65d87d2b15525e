"""cfneb_band_dots_noalloc against the band's own K4 reduction.

The entry point exists for code that cannot allocate GPU memory and has no workspace to give the library either: a
plug-in that lives inside somebody else's MD or optimiser loop and only ever sees the arrays it is handed, a process
whose device memory was committed in full when it started, a loop that cannot afford the device-wide stall a
cudaMalloc brings.  Its reduction scratch is therefore a fixed array inside libcfneb.so, shared by all calls on a GPU
and never cleared.  What can go wrong with that is exactly what these tests look at: the scratch address (a wrong one
faults or silently sums garbage), and contents left behind by an earlier call leaking into a later one -- so every
comparison is made on two calls in a row, on bands of different length, and the short band is run again after the
long one.  The reference is the existing path: cfneb_get_dots, i.e. reduce_kernel + the second stage of
scalar_kernel working in the handle's workspace.

Collected last on purpose (pytest -x stops at the first failure; a failure here must not hide the parity tests).
"""
import numpy as np
import pytest

from cfneb_workloads import build_workload

pytestmark = pytest.mark.gpu

TOL = 1e-10  # the relative tolerance of the force / energy parity tests (test_gpu_parity.TOL_FORCE)


def band_state(k, n_steps):
    """(X, G, v, dots) of configs[k] after n_steps iterations, all from the handle (the existing path)."""
    import paper_2510_16721_b200 as cf
    spec, pos, cells = build_workload(k)
    band = cf.CFNEB(pos, cells, cf.params_for(spec, cell_factor=0.0))
    band.step(n_steps)
    dots, _, G = band.get_dots()
    X, v = band.get_state()
    assert band.get_status().error == 0
    band.close()
    return X, G, v, dots


def scales(d):
    """|a| |b| for each of the ten products a.b (Cauchy-Schwarz): the size its rounding error is measured against."""
    pp, mm, gg, vv = d[:, 0], d[:, 1], d[:, 5], d[:, 9]
    s = lambda a, b: np.sqrt(a * b)
    return np.stack([pp, mm, s(pp, mm), s(gg, pp), s(gg, mm), gg, s(gg, vv), s(pp, vv), s(mm, vv), vv], axis=1)


def run_noalloc(X, G, v):
    """Upload, call the entry point with a caller-owned output, read back."""
    import torch
    import paper_2510_16721_b200 as cf
    dev = torch.device("cuda:0")
    Xd, Gd, vd = (torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (X, G, v))
    out = torch.full((X.shape[0], 10), float("nan"), dtype=torch.float64, device=dev)
    cf.band_dots_noalloc(Xd, Gd, vd, out)
    return out.cpu().numpy()


def check(got, ref):
    assert np.all(got[0] == 0.0) and np.all(got[-1] == 0.0)           # endpoint rows
    assert np.all(np.isfinite(got))
    err = np.abs(got[1:-1] - ref[1:-1]) / scales(ref[1:-1])
    assert err.max() < TOL, err.max()
    assert np.all(ref[1:-1, [0, 1, 5, 9]] > 0.0)                        # the band moved: v != 0, G != 0


def test_noalloc_dots_match_the_handle_on_consecutive_calls():
    short = band_state(0, 3)   # 31 atoms x 7 images: 102 components per image, most stage-1 blocks have no work
    long_ = band_state(2, 3)   # 2048 atoms x 16 images: 6153 components, several blocks and a ragged tail
    first = run_noalloc(*short[:3])
    check(first, short[3])
    second = run_noalloc(*long_[:3])          # second call, longer band: overwrites and extends the scratch in use
    check(second, long_[3])
    third = run_noalloc(*short[:3])           # back to the short band: slots of images 7..15 hold the long band's sums
    check(third, short[3])
    assert np.array_equal(first, third)       # fixed summation order, nothing inherited from the call in between
    assert np.array_equal(second, run_noalloc(*long_[:3]))


def test_noalloc_refuses_what_its_scratch_cannot_hold():
    import torch
    import paper_2510_16721_b200 as cf
    dev = torch.device("cuda:0")
    P = cf.NOALLOC_MAX_IMAGES + 1
    X = torch.zeros((P, 12), dtype=torch.float64, device=dev)
    out = torch.full((P, 10), 7.0, dtype=torch.float64, device=dev)
    with pytest.raises(cf.CfnebError) as e:
        cf.band_dots_noalloc(X, X, X, out)
    assert e.value.code == -7 and "CFNEB_NOALLOC_MAX_IMAGES" in str(e.value)
    assert bool((out == 7.0).all())           # nothing was launched
    # the largest band it accepts, against numpy on the same numbers
    rng = np.random.default_rng(11)
    Xh, Gh, vh = (rng.standard_normal((cf.NOALLOC_MAX_IMAGES, 5, 3)) for _ in range(3))
    got = run_noalloc(Xh, Gh, vh)
    tp, tm = (Xh[2:] - Xh[1:-1]).reshape(-1, 15), (Xh[1:-1] - Xh[:-2]).reshape(-1, 15)
    g, w = Gh[1:-1].reshape(-1, 15), vh[1:-1].reshape(-1, 15)
    dot = lambda a, b: np.einsum("pi,pi->p", a, b)
    ref = np.stack([dot(tp, tp), dot(tm, tm), dot(tp, tm), dot(g, tp), dot(g, tm), dot(g, g), dot(g, w), dot(tp, w),
                    dot(tm, w), dot(w, w)], axis=1)
    assert np.max(np.abs(got[1:-1] - ref) / scales(ref)) < TOL
    # a host pointer is refused, not dereferenced
    L = cf.lib()
    import ctypes
    host = np.zeros(3 * 12)
    hp = ctypes.c_void_p(host.ctypes.data)
    with torch.cuda.device(dev):
        rc = L.cfneb_band_dots_noalloc(hp, hp, hp, 3, 12, ctypes.c_void_p(out.data_ptr()), None)
    assert rc == -1 and b"not a device pointer" in L.cfneb_band_dots_noalloc_error()
