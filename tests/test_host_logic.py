"""Host-side logic of the CUDA library, checked on CPU through its host-only C-ABI entry points
(include/wave2d.h: wave2d_host_scalars, wave2d_host_plan).  No device is touched."""
import numpy as np
import pytest

from paper_2006_10142_b200 import binding as B


@pytest.mark.parametrize("gamma,ap,am", [(2.0, 0.125, 0.125), (2.0, 0.5, 0.4), (2.0, 1.0, 1.0), (1.0, 0.75, 0.6),
                                          (2.0, 18.0, 18.0), (2.0, 0.041, 0.03)])
def test_scalar_row_against_dense_lu(gamma, ap, am):
    """rho is the small root of ap z^2 - beta z + ap; (cp_p, inv_p) are the LU pivots of the Toeplitz matrix of
    (2.11)/(2.12) -- compared with an elimination of the dense matrix written out here."""
    row = B.host_scalars(gamma, ap, am, q=0.3)
    K = (row.size - 8) // 2
    beta = gamma + 2 * ap
    assert row[0] == am and row[1] == 0.3 and row[5] == ap and row[6] == beta
    assert row[4] == -(gamma + 2 * am)
    rho = row[2]
    assert 0 < rho < 1 and abs(ap * rho * rho - beta * rho + ap) <= 1e-15 * beta
    assert abs(row[3] * (beta - ap * rho) - 1.0) <= 1e-15
    n = K
    T = np.diag(np.full(n, beta)) + np.diag(np.full(n - 1, -ap), 1) + np.diag(np.full(n - 1, -ap), -1)
    U = T.copy()
    for p in range(1, n):                       # Gaussian elimination without pivoting (diagonally dominant)
        U[p] -= (U[p, p - 1] / U[p - 1, p - 1]) * U[p - 1]
    d = np.diag(U)
    np.testing.assert_allclose(row[8 + K:8 + 2 * K], 1.0 / d, rtol=1e-13)
    np.testing.assert_allclose(row[8:8 + K], ap / d, rtol=1e-13)
    assert abs(row[8 + K - 1] - rho) <= 1e-12 * rho or rho ** (2 * K) > 1e-12   # converges to rho at rate rho^(2p)


def _check_plan(n, nlines, unit, nw, sub, nbk, slots, fixed, frac):
    pieces, nstatic, cta_off = B.host_plan(n, nlines, unit, nw, sub, nbk, slots, fixed, frac)
    UT, NP = -(-n // unit), -(-nlines // 32)
    assert len(pieces) > 0 and 0 <= nstatic <= len(pieces)
    assert cta_off[0] == 0 and np.all(np.diff(cta_off) >= 0) and cta_off[-1] == nstatic
    cover = np.zeros((NP, UT), dtype=np.int32)
    for panel, ua, ub, nst in pieces:
        assert 0 <= panel < NP and 0 <= ua < ub <= UT and nst >= 1
        cover[panel, ua:ub] += 1
        gbase = max(ua - nbk, 0) // sub * sub                 # first unit the kernel streams for this piece
        end = gbase + nst * nw                                # one past the last
        assert gbase <= max(ua - nbk, 0)                      # carry warm-up: nbk units before the first output
        assert end >= min(ub + nbk, UT)                       # look-ahead: nbk units after the last output
        assert ua == 0 or ua - gbase >= nbk
        if ub < UT:
            assert end - nw < ub + nbk                        # no stage is streamed for nothing
    assert np.all(cover == 1)                                 # every (panel, unit) is written exactly once
    order = [(p, a) for p, a, _, _ in pieces]
    assert order == sorted(order)                             # handed out panel-major, left to right
    if fixed > 0:
        assert nstatic == 0
    return pieces, nstatic, cta_off


@pytest.mark.parametrize("n,nlines", [(4095, 4095), (16383, 16383), (8191, 2047), (2047, 8191), (1023, 1023),
                                        (127, 127), (1, 1), (7, 40), (300, 33)])
def test_plan_covers_every_unit_once(n, nlines):
    for unit, nw, sub in ((8, 16, 2), (8, 8, 1), (16, 16, 2), (32, 8, 1)):
        for nbk in (1, 3, 8):
            if nbk > nw:
                continue
            _check_plan(n, nlines, unit, nw, sub, nbk, 148, 0, 0.75)
            _check_plan(n, nlines, unit, nw, sub, nbk, 296, 0, 0.5)
            _check_plan(n, nlines, unit, nw, sub, nbk, 148, 3, 0.75)


def test_plan_config3_is_balanced():
    """config 3 (4095^2, 8-point units, 16 units per stage, nbk = 3, 148 CTAs): 75 % dealt out evenly, short tail."""
    pieces, nstatic, cta_off = _check_plan(4095, 4095, 8, 16, 2, 3, 148, 0, 0.75)
    share = np.array([pieces[cta_off[c]:cta_off[c + 1], 3].sum() for c in range(148)])
    assert share.min() >= 0.9 * share.max() and 18 <= share.max() <= 26      # ~ 0.75 * 4096 / 148 = 20.8 stages
    tail = pieces[nstatic:, 3]
    assert tail.max() <= 9 and tail.min() >= 1 and np.median(tail) <= 4      # short pieces for the dynamic part
    total = pieces[:, 3].sum()
    assert total <= 1.12 * 128 * 32                                          # cuts cost < 12 % extra stages


def test_host_entry_points_reject_bad_arguments():
    with pytest.raises(B.Wave2DError):
        B.host_scalars(2.0, -1.0, 0.5)
    with pytest.raises(B.Wave2DError):
        B.host_plan(100, 100, 8, 16, 2, 17, 148)     # carry series longer than a stage
    with pytest.raises(B.Wave2DError):
        B.host_plan(0, 100, 8, 16, 2, 3, 148)


@pytest.mark.parametrize("N,extent,tau,c,gamma,sigma", [(1024, 1.0, 1.0 / 1024, 1.5, 2.0, 0.5), (2048, 1.0, 1.0 / 8192, 1.3, 2.0, 0.5),
                                                        (150, 1.0, 1.0 / 150, 1.3, 2.0, 1.0), (4096, 1.0, 16.0 / 4096, 1.0, 1.0, 0.75)])
def test_decay_ratio_of_a_sweep(N, extent, tau, c, gamma, sigma):
    """wave2d_host_decay (what the row-block driver sizes its halo with): alpha+ = sigma tau^2 c / h^2, rho the small root of
    alpha+ z^2 - (gamma + 2 alpha+) z + alpha+ -- against the root written in its cancellation-free form, against the
    decay of a dense solve with a unit right-hand side at one end, and against the scalar row of the same alpha+."""
    rho = B.host_decay(N, extent, tau, c, gamma, sigma)
    h = extent / N
    ap = sigma * tau * tau * c / (h * h)
    beta = gamma + 2 * ap
    assert abs(rho - 2 * ap / (beta + np.sqrt(beta * beta - 4 * ap * ap))) <= 4e-16
    assert rho == B.host_scalars(gamma, ap, 0.3, 0.0)[2]
    n = 800                                    # long enough that the far end's reflection (rho^(2 (n - j))) is below rounding
    T = np.diag(np.full(n, beta)) + np.diag(np.full(n - 1, -ap), 1) + np.diag(np.full(n - 1, -ap), -1)
    x = np.linalg.solve(T, np.eye(n)[0])
    np.testing.assert_allclose(x[11:21] / x[10:20], rho, rtol=1e-9)     # the influence of an end decays like rho per point
    with pytest.raises(B.Wave2DError):
        B.host_decay(N, extent, tau, -1.0)
