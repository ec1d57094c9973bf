"""lgt_plaquette_action_noalloc: the entry point that allocates nothing (scratch in a file-scope __device__ array of the
library) against the existing path (lgt_action / lgt_plaquette on a handle) and the oracle, on two calls in a row.

Collected last on purpose (the suite runs with `pytest -x`): a failure here hides no other test.  Passes alone in a fresh
process and after the other tests -- it depends on no state they leave behind, and the array it shares is cleared per call.
"""
import numpy as np
import pytest

import oracle
from paper_2602_20516_b200 import synth

pytestmark = pytest.mark.gpu

BC = (1, 1, 1, -1)
TOL64 = 1e-11  # the fp64 tolerance of tests/test_gpu_parity.py
TOL32 = 2e-5   # its fp32 tolerance


@pytest.fixture(scope="module")
def lgt():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; the product path has no CPU fallback")
    from paper_2602_20516_b200 import lgt as m

    m.lib()
    return m


def existing_path(lgt, dims, beta, U, precision):
    lat = lgt.Lattice(dims, beta, 0.0, BC, precision)
    lat.set_links(U)
    S_g = lgt.lgt_action(lat.ctx)[0]
    plaq = lgt.lgt_plaquette(lat.ctx)
    lat.close()
    return S_g, plaq


def test_no_alloc_plaquette_action_matches_the_existing_path_twice_in_a_row(lgt):
    import torch

    # 1280 sites = 10 blocks of 128; then a ragged lattice (1350 sites: the last block is partly empty) with other links, so
    # that the second call finds the first call's partials and counter in the shared array
    cases = [((8, 4, 4, 10), 5.6, 0.3, 9101), ((5, 6, 5, 9), 6.0, 0.2, 9102)]
    out = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
    for dims, beta, eps, seed in cases:
        U = synth.warm_links(dims, eps, seed)
        S_ref, plaq_ref = existing_path(lgt, dims, beta, U, lgt.LGT_F64)
        Ud = torch.from_numpy(U).to(torch.complex128).cuda().contiguous()
        got = []
        for call in range(2):  # two calls in a row on the same stream, no clearing in between
            out.fill_(float("nan"))
            lgt.lgt_plaquette_action_noalloc(dims, beta, Ud, out, lgt.LGT_F64, 0, torch.cuda.current_stream().cuda_stream)
            torch.cuda.synchronize()
            got.append(out.cpu().numpy().copy())
        assert np.array_equal(got[0], got[1])  # fixed-order sums: the same bits
        S_g, plaq = got[0]
        assert abs(S_g - S_ref) <= TOL64 * abs(S_ref)
        assert abs(plaq - plaq_ref) <= TOL64 * abs(plaq_ref)
        S_or, plaq_or = oracle.gauge_action(dims, beta, U)
        assert abs(S_g - S_or) <= TOL64 * abs(S_or) and abs(plaq - plaq_or) <= TOL64 * abs(plaq_or)
        # fp32 links, sums in double: against the existing fp32 path
        S32_ref, plaq32_ref = existing_path(lgt, dims, beta, U, lgt.LGT_F32)
        U32 = Ud.to(torch.complex64).contiguous()
        for call in range(2):
            out.fill_(float("nan"))
            lgt.lgt_plaquette_action_noalloc(dims, beta, U32, out, lgt.LGT_F32, 0, torch.cuda.current_stream().cuda_stream)
            torch.cuda.synchronize()
            S32, plaq32 = out.cpu().numpy()
            assert abs(plaq32 - plaq32_ref) <= TOL32 * abs(plaq32_ref)
            assert abs(plaq32 - plaq_ref) <= TOL32 * abs(plaq_ref)
            assert abs(S32 - S32_ref) <= TOL32 * 6 * synth.volume(dims) * beta


def test_no_alloc_rejects_what_does_not_fit(lgt):
    import torch

    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    U = torch.zeros(16 * 4 * 9, dtype=torch.complex128, device="cuda")
    too_big = (256, 256, 256, 2)  # 2^25 sites > LGT_NOALLOC_MAX_SITES; rejected before anything is read
    assert 256 * 256 * 256 * 2 > lgt.LGT_NOALLOC_MAX_SITES
    with pytest.raises(lgt.LgtError) as e:
        lgt.lgt_plaquette_action_noalloc(too_big, 5.6, U, out)
    assert e.value.code == lgt.LGT_EINVAL and "LGT_NOALLOC_MAX_SITES" in str(e.value)
    with pytest.raises(lgt.LgtError):
        lgt.lgt_plaquette_action_noalloc((2, 2, 2, 2), 5.6, None, out)
    with pytest.raises(lgt.LgtError):
        lgt.lgt_plaquette_action_noalloc((2, 2, 2, 0), 5.6, U, out)
    with pytest.raises(lgt.LgtError):
        lgt.lgt_plaquette_action_noalloc((2, 2, 2, 2), 5.6, U, out, precision=7)
