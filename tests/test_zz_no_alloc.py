"""bh_direct_noalloc (include/bh.h): the direct sum of Eq. 2 with its scratch in a file-scope static
__device__ array of libbh -- an entry point that allocates nothing, for callers that cannot call cudaMalloc.

Checked against the EXISTING path (bh_build + bh_potential_direct, which keeps the same packed copy of the cells in
memory its context allocates) within the bar the direct-sum tests use (1e-12 relative, tests/test_gpu_parity.py;
the two paths add the same terms in different orders), on two calls in a row that share the static array -- the
second smaller than the first, so records the first call left behind lie beyond its n.  This file is collected last
on purpose (pytest -x: a failure here hides nothing) and passes alone as well as after the others.
"""
import numpy as np
import pytest

import bh_workloads as wl

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

TOL = 1e-12


@pytest.fixture(scope="module")
def bh():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_1509_07370_b200 as pkg
    return pkg


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()


def _existing(bh, w):
    ctx = bh.Context(0)
    ctx.build(_dev(w.x), _dev(w.y), _dev(w.z), _dev(w.m), w.cube)
    ref = ctx.potential_direct(w.G).cpu().numpy()
    ctx.close()
    return ref


def _rel(phi, ref):
    nz = ref != 0
    assert np.all(phi[~nz] == 0.0)
    return float(np.max(np.abs(phi[nz] - ref[nz]) / np.abs(ref[nz]))) if nz.any() else 0.0


def test_two_calls_in_a_row_equal_the_existing_path(bh):
    w1 = wl.random_points(4099, seed=2)                                   # several tiles + a ragged tail
    w2 = wl.with_duplicates(wl.clustered_points(3000, seed=3), 40, seed=4)   # smaller, with zero-distance pairs
    refs = [_existing(bh, w) for w in (w1, w2)]
    ins = [[_dev(a) for a in (w.x, w.y, w.z, w.m)] for w in (w1, w2)]
    outs = [torch.full((w.n,), float("nan"), dtype=torch.float64, device="cuda") for w in (w1, w2)]
    torch.cuda.synchronize()
    # both calls back to back on one stream, nothing in between: the second reuses the array the first filled
    bh.direct_noalloc(*ins[0], G=w1.G, out=outs[0])
    free_before = torch.cuda.mem_get_info()[0]
    bh.direct_noalloc(*ins[1], G=w2.G, out=outs[1])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before                    # the call took no device memory
    for w, out, ref in zip((w1, w2), outs, refs):
        phi = out.cpu().numpy()
        assert np.all(np.isfinite(phi))
        err = _rel(phi, ref)
        print(f"bh_direct_noalloc {w.name}: n={w.n} max rel {err:.2e} vs bh_potential_direct")
        assert err <= TOL
    # and once more with the first input: the same bits as its first call (the array keeps no state that matters)
    again = bh.direct_noalloc(*ins[0], G=w1.G).cpu().numpy()
    assert np.array_equal(again, outs[0].cpu().numpy())


def test_on_a_side_stream_and_at_the_limit(bh):
    n = bh.NOALLOC_MAX_N
    w = wl.random_points(n, seed=11)
    ref = _existing(bh, w)
    d = [_dev(a) for a in (w.x, w.y, w.z, w.m)]
    out = torch.empty(n, dtype=torch.float64, device="cuda")
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    bh.direct_noalloc(*d, G=w.G, out=out, stream=st)
    st.synchronize()
    assert _rel(out.cpu().numpy(), ref) <= TOL


def test_rejects_what_does_not_fit(bh):
    n = bh.NOALLOC_MAX_N + 1
    d = [torch.zeros(n, dtype=torch.float64, device="cuda") for _ in range(4)]
    out = torch.full((n,), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(bh.BHError) as ei:
        bh.direct_noalloc(*d, out=out)
    assert ei.value.code == -5 and "BH_NOALLOC_MAX_N" in str(ei.value)    # BH_ERR_TOO_LARGE, and it says why
    torch.cuda.synchronize()
    assert bool((out == 7.0).all())                                       # nothing was launched
    empty = [torch.empty(0, dtype=torch.float64, device="cuda") for _ in range(5)]
    bh.direct_noalloc(*empty[:4], out=empty[4])                           # n = 0 is fine
    one = wl.random_points(1, seed=9)
    phi = bh.direct_noalloc(*[_dev(a) for a in (one.x, one.y, one.z, one.m)]).cpu().numpy()
    assert phi.shape == (1,) and phi[0] == 0.0                            # a lone cell has no partner
