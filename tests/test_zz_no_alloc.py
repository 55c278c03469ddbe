"""dh_conserved_sums_noalloc (include/diffhydro.h; csrc/noalloc.cu): the conserved-sums diagnostic with its scratch in a
static device array -- no context, no allocation -- against the existing dh_conserved_sums on the same arrays, two calls
in a row (the second one finds the scratch as the first left it), plus the size limit.  Collected last on purpose: the
suite runs with pytest -x."""
import ctypes as C

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def api():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2502_02294_b200 import api
    return api


def _scale(gas, w, m_p):
    """sum |x| per output: what a relative bound on a sum of signed numbers refers to."""
    g = gas.double().abs().sum(dim=(1, 2, 3)).cpu().numpy()[:5]
    p = m_p * w.double().abs().sum(dim=1).cpu().numpy() if w is not None and w.numel() else np.zeros(3)
    return np.concatenate([g, p])


@pytest.mark.parametrize("N,nps", [(32, 32), (96, 40), (64, 0)])
def test_noalloc_sums_match_the_allocating_path_twice_in_a_row(api, W, N, nps):
    import torch
    # blocks take chunks of 32768 elements: 32^3 is one chunk, 96^3 is 27, 40^3 particles are one chunk and a ragged second
    gas, part = W.smooth_random_state(N, 11, amp=0.2, n_part_side=max(nps, 2))
    gas = torch.as_tensor(gas.astype(np.float32)).cuda()
    part = torch.as_tensor(part.astype(np.float32)).cuda() if nps else torch.zeros((6, 0), device="cuda")
    ctx = api.Context(N, float(N), 5.0 / 3.0, n_part_side=nps, static_mode=1, gravity_on=1 if nps else 0)
    m_p = (1.0 - 0.16) * N ** 3 / nps ** 3 if nps else 0.0          # the context's own: (1 - Omega_b / Omega_m) N^3 / n_part
    out = torch.full((8,), float("nan"), dtype=torch.float64, device="cuda")
    results = []
    for call in range(2):
        if call == 1:                                   # other numbers on the second call: nothing may carry over
            gas = (gas * 1.25 + 0.5).contiguous()
            part = (part * 0.5).contiguous()
        st = api.State(gas, part, 1.0)
        ref = ctx.dh_conserved_sums(st)
        api.dh_conserved_sums_noalloc(gas, part[3:6].contiguous() if nps else None, m_p, out)
        torch.cuda.synchronize()
        got = out.cpu().numpy().copy()
        assert np.all(np.isfinite(got))
        sc = _scale(gas, part[3:6] if nps else None, m_p)
        # both are fp64 sums of the same fp32 numbers in different orders: the bound of test_conserved_sums_diagnostic
        assert np.all(np.abs(got - ref) <= 1e-12 * sc + 1e-300), (call, got, ref)
        # and against numpy
        ref_np = np.concatenate([gas.double().sum(dim=(1, 2, 3)).cpu().numpy()[:5],
                                 m_p * part[3:6].double().sum(dim=1).cpu().numpy() if nps else np.zeros(3)])
        assert np.all(np.abs(got - ref_np) <= 1e-12 * sc + 1e-300)
        results.append(got)
        # the order of the additions is fixed: a repeat gives the same bits
        out.fill_(float("nan"))
        api.dh_conserved_sums_noalloc(gas, part[3:6].contiguous() if nps else None, m_p, out)
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy(), got)
    assert not np.array_equal(results[0], results[1])
    ctx.close()


def test_noalloc_ragged_cell_count_against_torch(api):
    """A cell count no mesh has (the context path cannot take it): 3 chunks and a tail of 1697 cells, then a single short
    chunk, on the same output array."""
    import torch
    gen = torch.Generator(device="cuda").manual_seed(5)
    x = torch.randn((5, 200000), device="cuda", generator=gen)
    out = torch.zeros(8, dtype=torch.float64, device="cuda")
    g = (C.c_void_p * 5)(*[x[k].data_ptr() for k in range(5)])
    for n in (100001, 777):
        assert api._lib.dh_conserved_sums_noalloc(g, n, None, 0, 0.0, C.c_void_p(out.data_ptr()), None) == 0
        torch.cuda.synchronize()
        ref = x[:, :n].double().sum(dim=1).cpu().numpy()
        sc = x[:, :n].double().abs().sum(dim=1).cpu().numpy()
        got = out.cpu().numpy()
        assert np.all(np.abs(got[:5] - ref) <= 1e-12 * sc) and np.all(got[5:] == 0.0)


def test_noalloc_rejects_sizes_beyond_its_static_scratch(api):
    import torch
    x = torch.zeros((5, 8, 8, 8), device="cuda")
    out = torch.zeros(8, dtype=torch.float64, device="cuda")
    g = (C.c_void_p * 5)(*[x[k].data_ptr() for k in range(5)])
    too_many = api.DH_NOALLOC_MAX_ELEMS + 1
    rc = api._lib.dh_conserved_sums_noalloc(g, too_many, None, 0, 1.0, C.c_void_p(out.data_ptr()), None)
    assert rc == -1
    msg = api._lib.dh_last_error().decode()
    assert "maximum" in msg and str(api.DH_NOALLOC_MAX_ELEMS) in msg
    w = (C.c_void_p * 3)(*[x[k].data_ptr() for k in range(3)])
    assert api._lib.dh_conserved_sums_noalloc(g, 512, w, too_many, 1.0, C.c_void_p(out.data_ptr()), None) == -1
    assert api._lib.dh_conserved_sums_noalloc(g, 0, None, 0, 1.0, C.c_void_p(out.data_ptr()), None) == -1
    assert api._lib.dh_conserved_sums_noalloc(g, 512, None, 0, 1.0, None, None) == -1
    # the limit itself is accepted by the argument check (not launched here: 5 x 512 MiB of input)
    torch.cuda.synchronize()
