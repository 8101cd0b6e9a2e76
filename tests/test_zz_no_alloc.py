"""mipwa_nll_parts_static (include/mipwa.h): the likelihood pieces (S, I, n_ev) with the kernel's scratch memory in the
library's file-scope device array, for callers that cannot call cudaMalloc.  Checked against the existing path
(mipwa_nll_parts_device on the recompute path, same kernel with the context's own buffers) and against the oracle (O7),
on two calls in a row with different parameters: the array keeps the first call's contents, the second must not see them.
Collected last on purpose (the name): the run uses pytest -x."""
import numpy as np
import pytest

from tests.helpers import make_case, nll_tol

pytestmark = pytest.mark.gpu


def _lib():
    from paper_1703_03284_b200 import binding
    return binding


@pytest.fixture(scope="module")
def case():
    return make_case(3, n_ev=30_011, n_norm=20_003)          # the bench model (a floating shape), ragged sizes


def _pieces(t):
    import torch
    torch.cuda.synchronize()
    return [float(v) for v in t.cpu()]


def test_static_scratch_matches_existing_path_twice_in_a_row(case):
    import torch
    c, o, data = case
    B = _lib()
    m = B.Mipwa(c.kin, c.knots, c.resonances)
    m.set_events(data[0], data[1]); m.set_norm_points(data[2], data[3], data[4])
    m.set_path(B.PATH_RECOMPUTE)
    got, ref = (torch.empty(3, dtype=torch.float64, device="cuda") for _ in range(2))
    with pytest.raises(B.MipwaError):                        # records not built yet: building them would allocate
        m.nll_parts_static(c.perturbed(0), got)
    m.nll(c.perturbed(0))                                    # builds the records (allocates)
    free_before = None
    for call, seed in enumerate((1, 2)):                     # two calls in a row, different parameters
        p = c.perturbed(seed)
        m.nll_parts_device(p, ref)
        S_r, I_r, n_r = _pieces(ref)
        got.fill_(-7.0)
        if call == 1:
            free_before = torch.cuda.mem_get_info()[0]
        m.nll_parts_static(p, got)
        S, Iv, n = _pieces(got)
        if call == 1:
            assert torch.cuda.mem_get_info()[0] == free_before   # no device allocation inside the call
        nll_ref, sl, integ = o.nll(p, *data, parts=True)
        tol = nll_tol(nll_ref, sl, integ, data[0].size)
        assert n == n_r == data[0].size
        assert abs(S - S_r) <= tol and abs(Iv - I_r) <= 1e-12 * I_r      # the existing path
        assert (S, Iv) == (S_r, I_r)                                      # same kernel, same grid: same bits
        assert abs((-S + n * np.log(Iv)) - nll_ref) <= tol                # the oracle
        assert abs(S - sl) <= tol and abs(Iv - integ) <= 1e-12 * integ
    # part of the GPU: another grid, another summation order, same tolerance; then the full grid again
    p = c.perturbed(3)
    m.nll_parts_device(p, ref)
    S_r, I_r, _ = _pieces(ref)
    nll_ref, sl, integ = o.nll(p, *data, parts=True)
    for blocks in (37, 0, 1, B.STATIC_MAX_BLOCKS):
        m.nll_parts_static(p, got, blocks=blocks)
        S, Iv, n = _pieces(got)
        assert abs(S - S_r) <= nll_tol(nll_ref, sl, integ, data[0].size) and abs(Iv - I_r) <= 1e-12 * I_r, blocks
    # the combine of the device route accepts the pieces like any others
    nll_d = m.combine_parts_device(got, 1)[0]
    assert abs(nll_d - nll_ref) <= nll_tol(nll_ref, sl, integ, data[0].size)
    m.close()


def test_static_scratch_refuses_what_does_not_fit(case):
    import torch
    c, _, data = case
    B = _lib()
    m = B.Mipwa(c.kin, c.knots, c.resonances)
    m.set_events(data[0], data[1]); m.set_norm_points(data[2], data[3], data[4])
    m.set_path(B.PATH_RECOMPUTE)
    p = c.perturbed(0)
    m.nll(p)
    out = torch.full((3,), -7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(B.MipwaError, match="static scratch"):
        m.nll_parts_static(p, out, blocks=B.STATIC_MAX_BLOCKS + 1)
    with pytest.raises(B.MipwaError):
        m.nll_parts_static(p, out, blocks=-1)
    with pytest.raises(B.MipwaError):
        m.nll_parts_static(p[:-1], out)
    torch.cuda.synchronize()
    assert out.cpu().tolist() == [-7.0, -7.0, -7.0]          # nothing was launched
    m.nll_parts_static(p, out)                               # and the entry point still works afterwards
    torch.cuda.synchronize()
    assert out[2].item() == data[0].size
    m.close()
