"""GPU edge cases of the C ABI: empty batches, odd vector counts, error codes, repeated calls, non-default stream."""
import numpy as np
import pytest

import oracle_problem
from gpu_common import make_west, random_vectors, relmax
from oracle import chi0 as ochi0

pytestmark = pytest.mark.gpu


def test_empty_batches_are_no_ops():
    import torch
    p = oracle_problem.build("cfg1")
    w, _ = make_west(p)
    x = torch.empty((0, w.n_g), dtype=torch.complex128, device="cuda")
    assert w.h_apply(x).shape == (0, w.n_g)
    assert w.fft3d(+1, x).shape[0] == 0
    dV = torch.empty((0, p.N, p.N, p.N), dtype=torch.float64, device="cuda")
    dn, _, st = w.chi0_apply(dV, [0.0], alpha_pv=p.alpha)
    assert dn.shape[1] == 0 and st["rc"] == 0
    w.close()


def test_error_codes():
    import torch
    import paper_2203_05623_b200 as wb
    with pytest.raises(wb.WestError) as e:
        wb.West(10.0, 25, 25, wb.WEST_FULL)                 # unsupported grid
    assert e.value.code == wb.binding.WEST_EINVAL
    with pytest.raises(wb.WestError) as e:
        wb.West(10.0, 100, 24, wb.WEST_FULL)                # grid too small for the sphere (aliasing)
    assert e.value.code == wb.binding.WEST_EINVAL
    w = wb.West(10.0, 25, 24, wb.WEST_FULL)
    x = torch.zeros((2, w.n_g), dtype=torch.complex128, device="cuda")
    with pytest.raises(wb.WestError) as e:
        w.h_apply(x)                                         # V_loc not set
    assert e.value.code == wb.binding.WEST_ESTATE
    dV = torch.zeros((1, 24, 24, 24), dtype=torch.float64, device="cuda")
    with pytest.raises(wb.WestError) as e:
        w.chi0_apply(dV, [0.0])
    assert e.value.code == wb.binding.WEST_ESTATE
    w.close()
    p = oracle_problem.build("cfg1")
    w, _ = make_west(p)
    with pytest.raises(wb.WestError) as e:
        w.chi0_apply(torch.zeros((1, p.N, p.N, p.N), dtype=torch.float64, device="cuda"), [0.5], alpha_pv=p.alpha)
    assert e.value.code == wb.binding.WEST_EINVAL            # omega > 0 needs WEST_GAMMA (reading R7)
    with pytest.raises(wb.WestError):
        w.chi0_apply(torch.zeros((1, p.N, p.N, p.N), dtype=torch.float64, device="cuda"), [-1.0], alpha_pv=p.alpha)
    w.close()


def test_constant_perturbation_gives_zero_response_and_linearity():
    import torch
    p = oracle_problem.build("mini2")
    w, _ = make_west(p)
    N = p.N
    const = np.full((1, N, N, N), 0.3)
    dV = np.concatenate([const, p.dV[:2], 2.0 * p.dV[:1] - 0.5 * p.dV[1:2]])
    dn, _, st = w.chi0_apply(torch.from_numpy(np.ascontiguousarray(dV)).cuda(), [0.0], tol=1e-12, alpha_pv=p.alpha)
    dn = dn.cpu().numpy()[0]
    scale = np.max(np.abs(dn[1]))
    assert np.max(np.abs(dn[0])) < 1e-12 * scale                                    # dV = const -> P_c(const * psi_v) = 0
    assert relmax(dn[3], 2.0 * dn[1] - 0.5 * dn[2]) < 1e-9                          # chi0 is linear
    w.close()


def test_repeated_calls_and_side_stream_give_identical_results():
    import torch
    import paper_2203_05623_b200 as wb
    p = oracle_problem.build("mini2")
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        mode = wb.WEST_GAMMA
        w = wb.West(p.L, p.n2max, p.N, mode, stream=st)
        w.set_vloc(torch.from_numpy(np.ascontiguousarray(p.vloc)).cuda())
        w.set_kb(torch.from_numpy(np.ascontiguousarray(p.beta[:, p.half])).cuda(), p.dcoef)
        c, cfull = random_vectors(p, 5, 3)
        x = torch.from_numpy(c).cuda()
        y1 = w.h_apply(x).clone()
        y2 = w.h_apply(x)
        st.synchronize()
    assert torch.equal(y1, y2)                                                      # H*psi is deterministic
    ref = (p.H @ cfull.T).T[:, p.half]
    assert relmax(y1.cpu().numpy(), ref) < 1e-9
    w.close()
