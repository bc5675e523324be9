"""hprmat_propagate_static: the propagation step (reading R16) for callers that may not allocate
device memory -- its workspace is a file-scope device array of the library (3 MiB per GPU, nch <= 128) instead of a caller's
buffer.  Checked against the existing path (hprmat_propagate with a workspace) on calls in a row that share the array, with
different sizes in between (the array keeps nothing a later call could see), against the oracle, and for the size limit.
Collected last on purpose (the suite runs with pytest -x).  Needs a B200 ("-m gpu")."""
import numpy as np
import pytest
import torch

import oracle
from paper_2512_11590_b200 import binding as hb

pytestmark = pytest.mark.gpu
DEV = "cuda"


def _case(nch, seed):
    """seeded sector matrices and R_in: O(1) complex entries, Rsec_LL + a_lo R_in safely invertible"""
    rng = np.random.default_rng(seed)
    def mat(diag):
        return rng.uniform(-1, 1, (nch, nch)) + 1j * rng.uniform(-1, 1, (nch, nch)) + diag * np.eye(nch)
    S = [[mat(2.0 * nch ** 0.5), mat(0.0)], [mat(0.0), mat(1.0)]]          # LL, LR / RL, RR
    R_in = mat(1.0)
    return S, R_in


def _col_major(a):
    """torch CUDA tensor whose memory is the column-major matrix a"""
    return torch.from_numpy(np.ascontiguousarray(a.T)).to(DEV)


def _run_both(nch, seed, a_lo=3.0, a_hi=7.5):
    S, R_in = _case(nch, seed)
    Rsec = torch.stack([_col_major(S[0][0]), _col_major(S[0][1]), _col_major(S[1][0]), _col_major(S[1][1])]).contiguous()
    Rin = _col_major(R_in)
    R_out = torch.full((nch, nch), float("nan"), dtype=torch.complex128, device=DEV)
    info = torch.full((1,), -7, dtype=torch.int32, device=DEV)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    hb.hprmat_propagate_static(a_lo, a_hi, Rin, Rsec, R_out, info)
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    got = R_out.cpu().numpy().T.copy()
    assert int(info.item()) == 0
    ref = hb.hprmat_propagate(a_lo, a_hi, Rin, Rsec).cpu().numpy().T.copy()      # the existing path, workspace per call
    orc = oracle.propagate(a_lo, a_hi, R_in, S)
    return got, ref, orc, free0 - free1


def test_static_scratch_propagation_matches_existing_path_on_calls_in_a_row():
    assert hb.hprmat_propagate_static_max_nch() == 128
    seen = set()
    for k, nch in enumerate([37, 128, 37, 128, 5, 128]):
        got, ref, orc, grew = _run_both(nch, seed=100 + k)
        scale = np.abs(ref).max()
        assert np.all(np.isfinite(got))
        # same kernels, same order, same data: identical to rounding (the tests' tolerance for this step is 1e-10)
        assert np.abs(got - ref).max() <= 1e-13 * scale, (k, nch, np.abs(got - ref).max() / scale)
        assert np.abs(got - orc).max() <= 1e-10 * np.abs(orc).max(), (k, nch)
        if nch in seen:
            # every kernel of this shape is loaded by now: the call must not have taken device memory
            assert grew <= 0, (k, nch, grew)
        seen.add(nch)


def test_static_scratch_rejects_sizes_beyond_its_limit():
    nch = 129
    S, R_in = _case(nch, 7)
    Rsec = torch.stack([_col_major(S[0][0]), _col_major(S[0][1]), _col_major(S[1][0]), _col_major(S[1][1])]).contiguous()
    R_out = torch.zeros((nch, nch), dtype=torch.complex128, device=DEV)
    info = torch.zeros(1, dtype=torch.int32, device=DEV)
    with pytest.raises(hb.HprmatError) as e:
        hb.hprmat_propagate_static(3.0, 7.5, _col_major(R_in), Rsec, R_out, info)
    assert e.value.code == hb.HPRMAT_ENOMEM and "128" in str(e.value)
    torch.cuda.synchronize()
    assert float(R_out.abs().max()) == 0.0        # nothing was launched
