"""Pins for the FP64 oracle against things other than itself: closed forms, textbook/library
routines, invariants, brute force on tiny inputs, and the full-matrix limit of the submatrix method
(the submatrix of a column whose pattern is full IS the matrix)."""
import os
from fractions import Fraction

import numpy as np
import pytest
import scipy.linalg as sla
import scipy.sparse as sp

import nolsm_inputs as gi
from nolsm_inputs.water import to_dense
import oracle.nolsm_oracle as orc

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ------------------------------------------------------------------ a0 neighbour lists
def _bruteforce_python(pos, box, rc):
    n = len(pos)
    out = []
    for j in range(n):
        row = []
        for i in range(n):
            d2 = 0
            for ax in range(3):
                d = int(pos[i][ax]) - int(pos[j][ax])
                L = int(box[ax])
                if d > L // 2:
                    d -= L
                elif d < -(L // 2):
                    d += L
                d2 += d * d
            if d2 <= rc * rc:
                row.append(i)
        out.append(row)
    return out


def test_neighbours_match_pure_python_bruteforce(tiny_system):
    s = tiny_system
    ref = _bruteforce_python(s.pos_q.tolist(), s.box_q.tolist(), s.rc_q)
    rp, ci = orc.neighbour_list(s.pos_q, s.box_q, s.rc_q)
    for j in range(s.n_mol):
        assert ci[rp[j]:rp[j + 1]].tolist() == ref[j]
    # and the generator's stored pattern is that same list (H and S share it; PAPER.md:158 merge = identity)
    assert np.array_equal(rp, s.row_ptr) and np.array_equal(ci, s.col_idx)


def test_neighbours_symmetric_self_included_and_full_at_large_cutoff(tiny_system):
    s = tiny_system
    rp, ci = orc.neighbour_list(s.pos_q, s.box_q, s.rc_q)
    pairs = {(j, int(i)) for j in range(s.n_mol) for i in ci[rp[j]:rp[j + 1]]}
    assert all((i, j) in pairs for (j, i) in pairs)
    assert all((j, j) in pairs for j in range(s.n_mol))
    # r_c >= L*sqrt(3)/2 (half the box diagonal) -> every molecule is everyone's neighbour
    rc_full = int(np.ceil(np.sqrt(3.0) / 2.0 * s.box_q[0])) + 1
    rp2, ci2 = orc.neighbour_list(s.pos_q, s.box_q, rc_full)
    assert np.array_equal(np.diff(rp2), np.full(s.n_mol, s.n_mol))
    assert np.array_equal(ci2.reshape(s.n_mol, s.n_mol), np.tile(np.arange(s.n_mol), (s.n_mol, 1)))


def test_neighbour_counts_match_continuum_estimate():
    # 4/3 pi r^3 rho molecules in a ball: 8 A -> 71.6 ; lattice + jitter gives ~80 (SURVEY table)
    s = gi.make_water_system(512, 8.0)
    m = np.diff(s.row_ptr)
    assert 70 <= m.mean() <= 90 and m.min() >= 60 and m.max() <= 100


def test_index_set_order():
    idx = orc.index_set(np.array([2, 5, 7]))
    assert idx.tolist() == [12, 13, 14, 15, 16, 17, 30, 31, 32, 33, 34, 35, 42, 43, 44, 45, 46, 47]


# ------------------------------------------------------------------ a1 submatrix construction
def test_dense_submatrix_equals_sparse_slicing(tiny_system):
    s = tiny_system
    n = s.n_mol * 6
    for val in (s.h_val, s.s_val):
        m = sp.bsr_matrix((val.astype(np.float64), s.col_idx, s.row_ptr), shape=(n, n)).tocsr()
        for j in (0, 7, 31):
            nb = s.col_idx[s.row_ptr[j]:s.row_ptr[j + 1]]
            idx = orc.index_set(nb)
            ref = m[idx][:, idx].toarray()
            got = orc.dense_submatrix(s.row_ptr, s.col_idx, val, nb)
            assert np.array_equal(ref, got)
            # not every neighbour pair of j is itself a stored pair -> genuine zeros appear
    nb = s.col_idx[s.row_ptr[0]:s.row_ptr[1]]
    sub = orc.dense_submatrix(s.row_ptr, s.col_idx, s.s_val, nb)
    assert (sub == 0).mean() > 0.05


# ------------------------------------------------------------------ Eq. 9-10 Newton-Schulz
def test_newton_schulz_scalar_closed_form():
    rows = [l.split() for l in open(os.path.join(GOLD, "ns_scalar_sequence.txt")) if not l.startswith("#")]
    exact = {int(k): Fraction(int(a), int(b)) for k, a, b in rows}
    # independent re-derivation of the golden rationals
    x = Fraction(1, 2)
    for k in range(4):
        assert x == exact[k]
        x = Fraction(1, 2) * x * (3 - x * x)
    # the oracle's matrix iteration on diag(0.5, -0.5) must reproduce them (sign is odd)
    for k in range(4):
        xk = orc.newton_schulz_sign(np.diag([0.5, -0.5]), k)
        assert abs(xk[0, 0] - float(exact[k])) < 1e-15 and abs(xk[1, 1] + float(exact[k])) < 1e-15
        assert xk[0, 1] == 0 and xk[1, 0] == 0
    # decimals quoted in SURVEY.md 8(c): 0.6875, 0.868774414062, 0.975299630819
    assert abs(float(exact[2]) - 0.868774414062) < 1e-12 and abs(float(exact[3]) - 0.975299630819) < 1e-12
    # from x0 = 0.05 ten iterations are needed to reach |x^2-1| < 1e-2
    x, k = 0.05, 0
    while abs(x * x - 1) >= 1e-2:
        x, k = 0.5 * x * (3 - x * x), k + 1
    assert k == 10
    _, res = orc.newton_schulz_sign(np.array([[0.05]]), 12, history=True)
    assert (res[:10] >= 1e-2).all() and res[10] < 1e-2


def test_newton_schulz_sign_converges_to_construction_and_quadratically():
    a, q, lam = gi.make_gapped_symmetric(48, seed=3)
    a = (q * lam) @ q.T
    exact = orc.sign_by_construction(q, lam)
    x, res = orc.newton_schulz_sign(a, 14, scale=np.abs(lam).max(), history=True)
    assert np.abs(x - exact).max() < 1e-12
    tail = res[(res < 1e-1) & (res > 1e-7)]
    # per eigenvalue e = x^2-1 maps to e' = 3/4 e^2 + O(e^3); with r = rms(e): 3/4 r^2 <= r' <= 3/4 sqrt(n) r^2
    for r0, r1 in zip(res[:-1], res[1:]):
        if 1e-6 < r0 < 3e-2:
            assert 0.74 * r0 * r0 < r1 < 0.77 * np.sqrt(48) * r0 * r0
    assert len(tail) >= 1
    # every iterate commutes with A
    x5 = orc.newton_schulz_sign(a, 5, scale=np.abs(lam).max())
    assert np.abs(x5 @ a - a @ x5).max() < 1e-13


def test_sign_by_construction_matches_library_signm():
    a, q, lam = gi.make_gapped_symmetric(24, seed=5)
    a64 = (q * lam) @ q.T
    ref = sla.signm(a64)
    assert np.abs(orc.sign_by_construction(q, lam) - ref).max() < 1e-10


# ------------------------------------------------------------------ Eq. 15-17 inverse
def test_newton_schulz_inverse_limits(tiny_system):
    s = tiny_system
    nb = s.col_idx[s.row_ptr[3]:s.row_ptr[4]]
    ssub = orc.dense_submatrix(s.row_ptr, s.col_idx, s.s_val, nb)
    c = np.abs(ssub).sum(axis=1).max()           # >= lambda_max
    sinv, z, y, res = orc.newton_schulz_inverse(ssub, 30, scale=c, history=True)
    assert np.abs(sinv - np.linalg.inv(ssub)).max() < 1e-12
    assert np.abs(y - sla.sqrtm(ssub / c)).max() < 1e-12          # Y -> Y0^{1/2}
    assert np.abs(z @ z @ (ssub / c) - np.eye(len(ssub))).max() < 1e-12   # Z -> Y0^{-1/2}
    assert np.abs(y @ z - np.eye(len(ssub))).max() < 1e-12
    # invariant Y_k = Y0 Z_k at every k
    for k in (1, 3):
        _, zk, yk = orc.newton_schulz_inverse(ssub, k, scale=c)
        assert np.abs(yk - (ssub / c) @ zk).max() < 1e-14
    assert res[0] > res[5] > res[-1]
    # 1x1: S = 4 -> inverse 1/4 whatever the (valid) scale
    sinv1, _, _ = orc.newton_schulz_inverse(np.array([[4.0]]), 40, scale=5.0)
    assert abs(sinv1[0, 0] - 0.25) < 1e-14


# ------------------------------------------------------------------ readings 5, 7, 11: scalings and early stop
def test_scaled_starts_stay_inside_the_convergence_intervals(tiny_system):
    """DESIGN.md readings 5 and 7.  Eq. 9 acts on an eigenvalue as x -> x(3 - x^2)/2, which converges to
    sign(x) exactly for 0 < |x| < sqrt(3); Eq. 16 acts on an eigenvalue of Z_k Y_k as v -> v(3 - v)^2/4, which
    converges to 1 for 0 < v < 3.  So X0 = 1.5 A/bound and Y0 = 2 S/bound (bound >= spectral radius) are
    valid starts, give the results of the unit scaling, and need no more iterations than it."""
    xs = np.array([-1.5, -1.0, -0.3, 0.05, 0.8, 1.5, 1.7])
    for _ in range(60):
        xs = 0.5 * xs * (3.0 - xs * xs)
    assert np.abs(xs - np.sign(xs)).max() < 1e-12
    x_out = 1.75                                   # beyond sqrt(3): leaves the basin (sign flips)
    for _ in range(60):
        x_out = 0.5 * x_out * (3.0 - x_out * x_out)
    assert not abs(x_out - 1.0) < 1e-6
    vs = np.array([0.05, 0.5, 1.0, 1.5, 2.0, 2.9])
    for _ in range(80):
        vs = 0.25 * vs * (3.0 - vs) ** 2
    assert np.abs(vs - 1.0).max() < 1e-12

    s = tiny_system
    nb = s.col_idx[s.row_ptr[5]:s.row_ptr[6]]
    ssub = orc.dense_submatrix(s.row_ptr, s.col_idx, s.s_val, nb)
    hsub = orc.dense_submatrix(s.row_ptr, s.col_idx, s.h_val, nb)
    n = len(ssub)
    a = np.linalg.solve(ssub, hsub) + 0.85 * np.eye(n)
    lam, v = orc.generalized_eig(hsub, ssub)
    ref = orc.sign_from_eig(lam, v, ssub, -0.85)
    bound = np.sqrt(np.abs(a).sum(0).max() * np.abs(a).sum(1).max())
    assert bound >= np.abs(lam + 0.85).max()
    x1, r1 = orc.newton_schulz_sign(a, 40, scale=bound, history=True)
    x2, r2 = orc.newton_schulz_sign(a, 40, scale=bound / 1.5, history=True)
    x3 = orc.newton_schulz_sign(a, 60, scale=np.abs(lam + 0.85).max() / 1.5)      # |x|_max = 1.5 exactly
    for x in (x1, x2, x3):
        assert np.abs(x - ref).max() < 1e-9
    first = lambda r: int(np.argmax(r < 1e-2))
    assert first(r2) <= first(r1)

    sb = np.sqrt(np.abs(ssub).sum(0).max() * np.abs(ssub).sum(1).max())
    inv = np.linalg.inv(ssub)
    i1, _, _, q1 = orc.newton_schulz_inverse(ssub, 40, scale=sb, history=True)
    i2, _, _, q2 = orc.newton_schulz_inverse(ssub, 40, scale=sb / 2, history=True)
    i3, _, _ = orc.newton_schulz_inverse(ssub, 60, scale=np.linalg.eigvalsh(ssub)[-1] / 2)   # v_max = 2 exactly
    for i in (i1, i2, i3):
        assert np.abs(i - inv).max() < 1e-10
    first3 = lambda r: int(np.argmax(r < 3e-3))
    assert first3(q2) <= first3(q1)


def test_inverse_residual_recurrence_and_refined_early_stop(tiny_system):
    """Reading 11.  With E_k = I - Z_k Y_k, Eq. 16 gives E_{k+1} = 3/4 E_k^2 + 1/4 E_k^3 exactly (V_{k+1} is a
    polynomial in V_k).  Taking Z_k at the first r_k < 3e-3 WITHOUT finishing the iteration, S0 = Z_k^2/s has a
    relative error of about 2 r_k, and one Newton step S0 + S0 (I - S S0) squares it."""
    s = tiny_system
    nb = s.col_idx[s.row_ptr[9]:s.row_ptr[10]]
    ssub = orc.dense_submatrix(s.row_ptr, s.col_idx, s.s_val, nb)
    n = len(ssub)
    eye = np.eye(n)
    c = 0.5 * max(1.0, np.sqrt(np.abs(ssub).sum(0).max() * np.abs(ssub).sum(1).max()))
    prev = None
    for k in range(0, 6):
        _, zk, yk = orc.newton_schulz_inverse(ssub, k, scale=c)
        e = eye - zk @ yk
        if prev is not None:
            assert np.abs(e - (0.75 * prev @ prev + 0.25 * prev @ prev @ prev)).max() < 1e-13
        prev = e
    _, _, _, res = orc.newton_schulz_inverse(ssub, 12, scale=c, history=True)
    k_stop = int(np.argmax(res < 3e-3))
    assert 0 < k_stop < 8
    _, zk, _ = orc.newton_schulz_inverse(ssub, k_stop, scale=c)
    s0 = zk @ zk / c
    inv = np.linalg.inv(ssub)
    rel0 = np.linalg.norm(s0 - inv, 2) / np.linalg.norm(inv, 2)
    s1 = s0 + s0 @ (eye - ssub @ s0)
    rel1 = np.linalg.norm(s1 - inv, 2) / np.linalg.norm(inv, 2)
    assert rel0 < 4 * np.sqrt(n) * res[k_stop]          # ||E||_2 <= ||E||_F = sqrt(n) r_k
    assert rel1 <= (np.linalg.cond(ssub) * rel0) ** 2 and rel1 < 1e-4


def test_a_priori_bound_on_the_next_inverse_residual(tiny_system, mid_system_cpu):
    """Reading 11, a-priori stop: E_k = I - Z_k Y_k is symmetric (a polynomial in S), so ||E_k||_2 <= ||E_k||_1 = b and
    the recurrence above gives ||E_{k+1}||_2 <= 3/4 b^2 + 1/4 b^3 -- known BEFORE iteration k is finished.  When the
    bound passes, Z_{k+1} alone is what the stopping rule needs; checked on the oracle's iterates of two systems, with
    the iteration at which the CUDA path's tolerance (2e-2) is first met and the quality of the iterate it takes."""
    for system, j in ((tiny_system, 9), (mid_system_cpu, 100)):
        nb = system.col_idx[system.row_ptr[j]:system.row_ptr[j + 1]]
        ssub = orc.dense_submatrix(system.row_ptr, system.col_idx, system.s_val, nb)
        n = len(ssub)
        eye = np.eye(n)
        c = 0.5 * max(1.0, np.sqrt(np.abs(ssub).sum(0).max() * np.abs(ssub).sum(1).max()))
        first = None
        for k in range(0, 6):
            _, zk, yk = orc.newton_schulz_inverse(ssub, k, scale=c)
            _, zk1, yk1 = orc.newton_schulz_inverse(ssub, k + 1, scale=c)
            e, e1 = eye - zk @ yk, eye - zk1 @ yk1
            assert np.abs(e - e.T).max() < 1e-13
            b = np.abs(e).sum(0).max()
            bound = 0.75 * b * b + 0.25 * b ** 3
            assert np.linalg.norm(e, 2) <= b * (1 + 1e-12)
            assert np.linalg.norm(e1, 2) <= bound * (1 + 1e-9) + 1e-13   # + the FP64 rounding floor
            if first is None and bound <= 2e-2:
                first = k
                # the iterate taken: Z_{k+1}.  Everything is a polynomial in S, so I - S Z^2/s IS E_{k+1}: S0 = Z^2/s
                # has a relative residual of at most the bound in EVERY direction
                s0 = zk1 @ zk1 / c
                assert np.abs((eye - ssub @ s0) - e1).max() < 1e-12
                assert np.linalg.norm(eye - ssub @ s0, 2) <= bound * (1 + 1e-9) + 1e-13
        assert first is not None and 1 <= first <= 3


def test_refinements_of_the_operator_cube_the_inverse_error(mid_system_cpu):
    """Reading 11, FP32 mode of the whole path: with A0 any approximate inverse of S and F = I - A0 S, the iteration
    B_{r+1} = B_r + A0 (H - S B_r) from B_0 = A0 H has B - B_r = F^(r+1) B exactly (B = S^-1 H), and the same for the
    own columns V of S^-1.  With the iterate the a-priori stop takes at 1e-2, two refinements leave < 1e-6 |B|."""
    system, j = mid_system_cpu, 100
    nb = system.col_idx[system.row_ptr[j]:system.row_ptr[j + 1]]
    ssub = orc.dense_submatrix(system.row_ptr, system.col_idx, system.s_val, nb)
    hsub = orc.dense_submatrix(system.row_ptr, system.col_idx, system.h_val, nb)
    n = len(ssub)
    eye = np.eye(n)
    c = 0.5 * max(1.0, np.sqrt(np.abs(ssub).sum(0).max() * np.abs(ssub).sum(1).max()))
    k_stop = None
    for k in range(6):
        _, zk, yk = orc.newton_schulz_inverse(ssub, k, scale=c)
        b1 = np.abs(eye - zk @ yk).sum(0).max()
        if 0.75 * b1 * b1 + 0.25 * b1 ** 3 <= 1e-2:
            k_stop = k
            break
    assert k_stop is not None
    _, z, _ = orc.newton_schulz_inverse(ssub, k_stop + 1, scale=c)
    a0 = (z @ z / c).astype(np.float16).astype(np.float64)          # the CUDA path keeps A0 in FP16
    f = eye - a0 @ ssub
    assert np.linalg.norm(f, 2) <= 1e-2 + 2e-3                        # the bound + the FP16 rounding of A0
    b_exact = np.linalg.solve(ssub, hsub)
    v_exact = np.linalg.inv(ssub)[:, :6]
    br, vr = a0 @ hsub, a0[:, :6].copy()
    fp = f.copy()
    for r in range(3):
        assert np.abs((b_exact - br) - fp @ b_exact).max() < 1e-12
        assert np.abs((v_exact - vr) - fp @ v_exact).max() < 1e-12
        br = br + a0 @ (hsub - ssub @ br)
        vr = vr + a0 @ (eye[:, :6] - ssub @ vr)
        fp = fp @ f
    b2 = a0 @ hsub
    for _ in range(2):
        b2 = b2 + a0 @ (hsub - ssub @ b2)
    assert np.abs(b2 - b_exact).max() < 1e-6 * np.abs(b_exact).max()


def test_lowdin_form_gives_the_same_density(tiny_solution, mid_system_cpu):
    """the symmetric Loewdin form S^-1/2 (1/2 (I - sign(S^-1/2 H S^-1/2 - mu I))) S^-1/2 is the density of
    the generalized problem (Eq. 12), and the thin-product route the CUDA path takes -- U = P~ Z[:, own],
    D[:, own] = Z U / s with Z = (S/s)^-1/2 -- reproduces its own columns."""
    sols = [tiny_solution["solutions"][7]]
    sols.append(orc.solve_molecule(mid_system_cpu.row_ptr, mid_system_cpu.col_idx, mid_system_cpu.h_val,
                                   mid_system_cpu.s_val, 100))
    for sol in sols:
        own = orc.own_position(sol.nbrs, sol.j)
        cols = np.arange(own * 6, own * 6 + 6)
        d_low = orc.density_columns_lowdin(sol.h_sub, sol.s_sub, cols, -0.85)
        assert np.abs(d_low - sol.density_columns(-0.85)).max() < 1e-10
        # the factored route, with an arbitrary scale s
        s_scale = 0.5 * np.abs(sol.s_sub).sum(0).max()
        sl, sv = np.linalg.eigh(sol.s_sub / s_scale)
        z = (sv / np.sqrt(sl)) @ sv.T
        at = z @ sol.h_sub @ z / s_scale
        x = orc.newton_schulz_sign(at + 0.85 * np.eye(len(z)), 40,
                                   scale=np.sqrt(np.abs(at + 0.85 * np.eye(len(z))).sum(0).max() ** 2) / 1.5)
        u = 0.5 * (z[:, cols] - x @ z[:, cols])
        assert np.abs(z @ u / s_scale - sol.density_columns(-0.85)).max() < 1e-9


def test_rescaled_first_sign_iteration(tiny_solution, mid_system_cpu):
    """Reading 5, rescaled first iteration: (1) the factor keeps the spectrum of a X0 inside [-1.7, 1.7] (1.7 < sqrt 3); (2) the update
    a (3/2 - 1/2 a^2) X0 + 1/2 a^3 X0 E_0 IS Eq. 9 applied to a X0; (3) the iteration converges to the same sign
    function (the eigenvector construction); (4) it never needs more iterations than the plain one, and on a
    water-like submatrix scaled by the O(n^2) norm bound it needs one fewer."""
    sols = [tiny_solution["solutions"][7]]
    sols.append(orc.solve_molecule(mid_system_cpu.row_ptr, mid_system_cpu.col_idx, mid_system_cpu.h_val,
                                   mid_system_cpu.s_val, 100))
    fewer = 0
    for sol in sols:
        n = len(sol.s_sub)
        eye = np.eye(n)
        a = np.linalg.solve(sol.s_sub, sol.h_sub) + 0.85 * eye
        scale = np.sqrt(np.abs(a).sum(0).max() * np.abs(a).sum(1).max()) / 1.5
        x0 = a / scale
        al = orc.rescaled_first_step_factor(x0)
        rho = np.abs(np.linalg.eigvals(x0)).max()
        assert orc.RESCALE_TARGET < np.sqrt(3.0)
        assert 1.0 <= al <= 1.7 and al * rho <= 1.7 * (1 + 1e-12) and rho ** 2 <= np.abs(x0 @ x0).sum(0).max() * (1 + 1e-12)
        e0 = eye - x0 @ x0
        x1 = al * (1.5 - 0.5 * al * al) * x0 + 0.5 * al ** 3 * (x0 @ e0)
        assert np.abs(x1 - 0.5 * (al * x0) @ (3 * eye - (al * x0) @ (al * x0))).max() < 1e-13
        assert np.abs(orc.newton_schulz_sign_rescaled(a, 1, scale=scale) - x1).max() < 1e-14
        # same limit as the plain iteration and as the construction from the generalized eigenvectors
        x_res = orc.newton_schulz_sign_rescaled(a, 40, scale=scale)
        x_plain = orc.newton_schulz_sign(a, 40, scale=scale)
        sign_ref = eye - 2.0 * sol.density(-0.85) @ sol.s_sub          # sign(A) = I - 2 D S  (Eq. 12 solved for the sign)
        assert np.abs(x_res - x_plain).max() < 1e-9 and np.abs(x_res - sign_ref).max() < 1e-8
        _, r_res = orc.newton_schulz_sign_rescaled(a, 20, scale=scale, history=True)
        _, r_plain = orc.newton_schulz_sign(a, 20, scale=scale, history=True)
        k_res, k_plain = int(np.argmax(r_res < 1e-2)), int(np.argmax(r_plain < 1e-2))
        assert 0 < k_res <= k_plain
        fewer += k_plain - k_res
    assert fewer >= 1


def test_last_sign_update_folded_into_thin_products(tiny_system, tiny_solution):
    """Reading 9: with E_k = I - X_k^2, X_{k+1} V = X_k (V + 1/2 E_k V) for any thin V, so the own columns of
    D = 1/2 (I - X_{k+1}) S^-1 follow from X_k and E_k without forming X_{k+1}."""
    s = tiny_system
    sol = tiny_solution["solutions"][7]
    hsub, ssub = sol.h_sub, sol.s_sub
    n = len(ssub)
    a = np.linalg.solve(ssub, hsub) + 0.85 * np.eye(n)
    bound = np.sqrt(np.abs(a).sum(0).max() * np.abs(a).sum(1).max())
    k = 7
    xk = orc.newton_schulz_sign(a, k, scale=bound / 1.5)
    xk1 = orc.newton_schulz_sign(a, k + 1, scale=bound / 1.5)
    ek = np.eye(n) - xk @ xk
    own = orc.own_position(sol.nbrs, sol.j)
    v = np.linalg.inv(ssub)[:, own * 6:own * 6 + 6]
    folded = 0.5 * (v - xk @ (v + 0.5 * ek @ v))
    direct = 0.5 * (v - xk1 @ v)
    assert np.abs(folded - direct).max() < 1e-13
    # and once converged this is the oracle's D column block
    x30 = orc.newton_schulz_sign(a, 30, scale=bound / 1.5)
    assert np.abs(0.5 * (v - x30 @ v) - sol.density_columns(-0.85)).max() < 1e-9


def test_scaled_newton_schulz_start(tiny_solution):
    """gap_hint.  Scalar facts: for l <= x <= 1 and a = sqrt(3/(1+l+l^2)) the step
    g(x) = a x (3 - a^2 x^2)/2 maps both ends to the same value l' > plain step of l, stays in (0, 1], and a
    wrong (too large) l still converges.  Matrix fact: same sign(A) as the plain iteration in fewer steps."""
    for l in (0.02, 0.1, 0.4):
        a = np.sqrt(3.0 / (1.0 + l + l * l))
        g = lambda x: 0.5 * a * x * (3.0 - a * a * x * x)
        assert abs(g(l) - g(1.0)) < 1e-14 and g(l) > 0.5 * l * (3.0 - l * l)
        xs = np.linspace(l, 1.0, 2001)
        assert g(xs).min() >= g(l) - 1e-14 and g(xs).max() <= 1.0 + 1e-14
    x = np.array([[0.01]])                                   # hint ten times too large
    assert abs(orc.newton_schulz_sign_scaled(x, 40, 1.0, 0.1)[0, 0] - 1.0) < 1e-12
    sol = tiny_solution["solutions"][11]
    n = sol.n
    a = np.linalg.solve(sol.s_sub, sol.h_sub) + 0.85 * np.eye(n)
    ref = sol.sign(-0.85)
    scale = np.sqrt(np.abs(a).sum(0).max() * np.abs(a).sum(1).max()) / 1.5
    gap = np.abs(sol.lam + 0.85).min()
    res = lambda x: np.linalg.norm(x @ x - np.eye(n)) / np.sqrt(n)
    k_plain = next(k for k in range(1, 40) if res(orc.newton_schulz_sign(a, k, scale=scale)) < 1e-8)
    k_scaled = next(k for k in range(1, 40) if res(orc.newton_schulz_sign_scaled(a, k, scale, 0.9 * gap)) < 1e-8)
    assert k_scaled <= k_plain - 2
    xs, alphas = orc.newton_schulz_sign_scaled(a, k_scaled + 2, scale, 0.9 * gap, history=True)
    assert np.abs(xs - ref).max() < 1e-9
    assert alphas[0] == 1.0 and alphas[1] > 1.3 and alphas[-1] == 1.0 and np.all(alphas < np.sqrt(3.0))


# ------------------------------------------------------------------ Eq. 6 / 12 by eigenvectors
def test_sign_and_density_identities(tiny_solution):
    sol = tiny_solution["solutions"][5]
    mu = -0.85
    n = sol.n
    sg = sol.sign(mu)
    a = np.linalg.solve(sol.s_sub, sol.h_sub) - mu * np.eye(n)
    assert np.abs(sg @ sg - np.eye(n)).max() < 1e-11                       # sign^2 = I
    assert np.abs(sg @ a - a @ sg).max() < 1e-11                           # commutes with A
    d = sol.density(mu)
    assert np.abs(sg - (np.eye(n) - 2 * d @ sol.s_sub)).max() < 1e-11      # sign = I - 2 D S
    assert np.abs(d - 0.5 * (np.eye(n) - sg) @ np.linalg.inv(sol.s_sub)).max() < 1e-11   # Eq. 12 literally
    assert np.abs(d @ sol.s_sub @ d - d).max() < 1e-12                     # D S D = D
    assert np.abs(d - d.T).max() < 1e-14
    nocc = int((sol.lam < mu).sum())
    assert abs(np.trace(d @ sol.s_sub) - nocc) < 1e-10                     # tr(DS) = # occupied, an integer
    ev = np.sort(np.linalg.eigvals(sg).real)
    assert np.abs(ev[:nocc] + 1).max() < 1e-9 and np.abs(ev[nocc:] - 1).max() < 1e-9
    # the literal Newton-Schulz iteration (Eq. 9-10) reaches the same sign
    x = orc.newton_schulz_sign(a, 40, scale=1.05 * np.abs(np.linalg.eigvals(a)).max())
    assert np.abs(x - sg).max() < 1e-9
    # own columns / populations are consistent with the full D
    assert np.abs(sol.density_columns(mu) - d[:, sol.own]).max() < 1e-14
    q = 2 * (d @ sol.s_sub)[sol.own, sol.own].sum()
    assert abs(q - sol.population(mu)) < 1e-11
    assert abs(q - 8.0) < 0.05


def test_orthogonal_case_reduces_to_textbook_eigh():
    rng = np.random.default_rng(0)
    h = rng.standard_normal((20, 20))
    h = h + h.T
    lam, v = orc.generalized_eig(h, np.eye(20))
    w, u = np.linalg.eigh(h)
    assert np.abs(lam - w).max() < 1e-12
    mu = 0.1
    p_ref = u[:, w < mu] @ u[:, w < mu].T
    assert np.abs(orc.density_from_eig(lam, v, mu) - p_ref).max() < 1e-12
    assert np.abs(orc.sign_from_eig(lam, v, np.eye(20), mu) - sla.signm(h - mu * np.eye(20))).max() < 1e-9


# ------------------------------------------------------------------ whole method, limit case
def test_full_cutoff_limit_equals_full_matrix_diagonalisation():
    """With r_c >= half the box diagonal every submatrix is the whole matrix, so the submatrix
    method must reproduce the full-matrix projector (north_star pin)."""
    s = gi.make_water_system(32, 9.0)
    assert (np.diff(s.row_ptr) == 32).all()
    H, S = to_dense(s, "H"), to_dense(s, "S")
    lam, v = sla.eigh(H, S)
    nocc = 4 * s.n_mol
    mu = 0.5 * (lam[nocc - 1] + lam[nocc])
    d_full = v[:, :nocc] @ v[:, :nocc].T
    out = orc.solve_system(s, mu=mu)
    assert abs(out["n_electrons"] - 8 * s.n_mol) < 1e-9                    # tr(DS) = 4N exactly
    d_val = out["d_val"]
    for j in range(s.n_mol):
        for k in range(s.row_ptr[j], s.row_ptr[j + 1]):
            i = s.col_idx[k]
            assert np.abs(d_val[k] - d_full[6 * i:6 * i + 6, 6 * j:6 * j + 6]).max() < 1e-11
    assert np.abs(d_full @ S @ d_full - d_full).max() < 1e-12
    # block contraction equals the trace
    assert abs(orc.electron_count_blocks(s.row_ptr, s.col_idx, d_val, s.s_val) - 8 * s.n_mol) < 1e-9


def test_submatrix_result_close_to_full_matrix_at_finite_cutoff(tiny_system, tiny_solution):
    """At 6 A the submatrix D differs from the full-matrix D by a few 1e-3 (nearsightedness)."""
    s = tiny_system
    H, S = to_dense(s, "H"), to_dense(s, "S")
    lam, v = sla.eigh(H, S)
    nocc = 4 * s.n_mol
    d_full = v[:, :nocc] @ v[:, :nocc].T
    d_val = tiny_solution["d_val"]
    err = 0.0
    for j in range(s.n_mol):
        for k in range(s.row_ptr[j], s.row_ptr[j + 1]):
            i = s.col_idx[k]
            err = max(err, np.abs(d_val[k] - d_full[6 * i:6 * i + 6, 6 * j:6 * j + 6]).max())
    assert 1e-5 < err < 2e-2


# ------------------------------------------------------------------ a7 electron count and mu
def test_electron_count_staircase_and_bisection(tiny_system, tiny_solution):
    s, sols = tiny_system, tiny_solution["solutions"]
    assert orc.electron_count(sols, -1e9) == 0.0
    assert abs(orc.electron_count(sols, 1e9) - 12 * s.n_mol) < 1e-9       # all 6 orbitals x 2
    homo, lumo = orc.mu_plateau(sols, lambda x: 4 * len(x.nbrs))
    assert homo < lumo
    mus = np.linspace(homo + 1e-6, lumo - 1e-6, 7)
    ne = [orc.electron_count(sols, m) for m in mus]
    assert max(ne) - min(ne) < 1e-12                                       # constant on the gap plateau
    assert abs(ne[0] - 8 * s.n_mol) < 2e-3 * s.n_mol                      # plateau is N_e only approximately
    grid = np.linspace(-2.5, -0.3, 400)
    vals = np.array([orc.electron_count(sols, m) for m in grid])
    assert (np.diff(vals) > -1e-3).all()                                   # monotone up to Mulliken wiggles
    mu, n_e, steps, trace = bisect_mu = orc.bisect_mu(sols, s.n_electrons, -3.0, 0.0)
    assert [t[0] for t in trace] == [-1.5, -0.75] and steps == 2
    assert homo < mu < lumo and abs(n_e - s.n_electrons) <= 1e-3 * s.n_mol
    # block contraction on the stored D equals the sum of populations
    nb = orc.electron_count_blocks(s.row_ptr, s.col_idx, tiny_solution["d_val"], s.s_val)
    assert abs(nb - tiny_solution["n_electrons"]) < 1e-9
    # per-molecule populations close to 8
    q = np.array([x.population(mu) for x in sols])
    assert np.abs(q - 8).max() < 0.03


def test_density_blocks_layout(tiny_system, tiny_solution):
    """Block k of row j of D is D(col_idx[k], j): rows of the neighbour, own columns of j."""
    s = tiny_system
    sol = tiny_solution["solutions"][9]
    mu = tiny_solution["mu"]
    d = sol.density(mu)
    a = 4
    k = s.row_ptr[9] + a
    assert np.abs(tiny_solution["d_val"][k] - d[6 * a:6 * a + 6][:, sol.own]).max() < 1e-14


# ------------------------------------------------------------------ generator sanity (inputs)
def test_generator_properties(tiny_system):
    s = tiny_system
    S, H = to_dense(s, "S"), to_dense(s, "H")
    assert np.array_equal(S, S.T) and np.array_equal(H, H.T)
    w = np.linalg.eigvalsh(S)
    assert w[0] > 0.3 and w[-1] < 2.5                                     # SPD without any shift
    lam = sla.eigh(H, S, eigvals_only=True)
    nocc = 4 * s.n_mol
    assert lam[nocc] - lam[nocc - 1] > 0.2                                 # gap at 4 occupied per molecule
    assert (s.box_q % 2 == 0).all() and s.pos_q.min() >= 0 and (s.pos_q < s.box_q).all()
    s2 = gi.make_water_system(32, 6.0)
    assert np.array_equal(s2.pos_q, s.pos_q) and np.array_equal(s2.h_val, s.h_val)   # seeded
    s3 = gi.make_water_system(32, 6.0, seed=1)
    assert not np.array_equal(s3.pos_q, s.pos_q)


def test_microbench_matrix_properties():
    a, q, lam = gi.make_gapped_symmetric(64, seed=11)
    assert np.abs(q.T @ q - np.eye(64)).max() < 1e-12
    assert 0.05 <= np.abs(lam).min() and np.abs(lam).max() <= 1.0 and (lam > 0).any() and (lam < 0).any()
    assert np.abs(np.linalg.eigvalsh(a.astype(np.float64)) - np.sort(lam)).max() < 1e-6
    assert gi.microbench_batch(256) == 512 and gi.microbench_batch(1024) == 8 and gi.microbench_batch(4096) == 1


def test_energy_weighted_density_and_energy_pins(tiny_system, tiny_solution):
    """Eq. 7, 8, 11, 13.  Pins: (i) with V^T S V = I and H V = S V Lambda, D H D collapses to
    V_occ Lambda_occ V_occ^T, a different formula from the triple product the oracle evaluates;
    (ii) tr(W_j S_j) = tr(D_j H_j) = sum of the occupied eigenvalues of the submatrix; (iii) at full
    cutoff every submatrix is the whole system, so the block sum of Eq. 11 equals the sum of the
    occupied eigenvalues of the full generalized problem (textbook band energy)."""
    mu = tiny_solution["mu"]
    for s in tiny_solution["solutions"][:6]:
        occ = s.lam < mu
        w = s.energy_weighted(mu)
        closed = (s.v[:, occ] * s.lam[occ]) @ s.v[:, occ].T
        assert np.abs(w - closed).max() < 1e-12
        assert abs(np.trace(w @ s.s_sub) - s.lam[occ].sum()) < 1e-11
        assert abs(np.trace(s.density(mu) @ s.h_sub) - s.lam[occ].sum()) < 1e-11
        assert np.abs(w - w.T).max() < 1e-12
        assert np.array_equal(s.energy_weighted_columns(mu), w[:, s.own])
    # full cutoff: block contraction of Eq. 11 against the full-matrix eigenvalues
    full = gi.make_water_system(32, 9.0)
    sol = orc.solve_system(full, mu=-0.85)
    d = orc.density_blocks(sol["solutions"], full.row_ptr, -0.85)
    e_blocks = orc.electronic_energy_blocks(full.row_ptr, full.col_idx, d, full.h_val)
    lam = sla.eigh(to_dense(full, "H"), to_dense(full, "S"), eigvals_only=True)
    assert abs(e_blocks - lam[lam < -0.85].sum()) < 1e-9
    # and the own columns of W in the store layout give tr(W S) = E when contracted like tr(D S)
    w_blocks = orc.energy_weighted_blocks(sol["solutions"], full.row_ptr, -0.85)
    assert abs(0.5 * orc.electron_count_blocks(full.row_ptr, full.col_idx, w_blocks, full.s_val) - e_blocks) < 1e-9


# ------------------------------------------------------------------ two-centre element model (row f2)
def _hand_model():
    # the literal constants of BASELINE.json configs[0] / DESIGN.md section 3, typed here (not imported)
    return dict(unit_per_grid=1.0 / 65536.0,
                site_offset=[[0.0, 0.0, 0.0], [0.757, 0.586, 0.0], [-0.757, 0.586, 0.0]],
                orb_site=[0, 0, 0, 0, 1, 2], orb_energy=[-1.0, -1.0, -1.0, -1.0, -0.5, -0.5],
                s_ampl=0.3, h_ampl=-0.2, h_len=1.5)


def test_two_centre_model_hand_values():
    """Pins of oracle.two_centre_block on numbers worked out by hand (decimal literals below):
    an intermolecular pair at the integer distance 3 A, the on-site block, the orbital -> site map, and
    a pair that is only close across the periodic boundary."""
    g = 65536
    box = np.array([40 * g, 40 * g, 40 * g], dtype=np.int32)
    pos = np.array([[0, 0, 0], [3 * g, 0, 0], [39 * g, 0, 0]], dtype=np.int32)   # molecule 2 is 1 A from 0 across the wall
    m = _hand_model()
    h, s = orc.two_centre_block(pos, box, 0, 1, m)
    # O(0) - O(1): r = 3:  S = 0.3 exp(-4.5),  H = -0.2 exp(-2)
    assert abs(s[0, 0] - 0.3 * 0.011108996538242306) < 1e-15
    assert abs(h[0, 0] - (-0.2 * 0.1353352832366127)) < 1e-15
    assert np.all(s[:4, :4] == s[0, 0]) and np.all(h[:4, :4] == h[0, 0])        # the four O-site orbitals share the site
    # O(0) - H1(1): d = (0,0,0) - (3.757, 0.586, 0): r^2 = 14.115049 + 0.343396 = 14.458445
    assert abs(s[0, 4] - 0.3 * np.exp(-0.5 * 14.458445)) < 1e-15
    assert abs(h[0, 4] - (-0.2 * np.exp(-np.sqrt(14.458445) / 1.5))) < 1e-15
    # O(0) - H2(1): d = -(3 - 0.757, 0.586, 0): r^2 = 2.243^2 + 0.586^2 = 5.031049 + 0.343396 = 5.374445
    assert abs(s[0, 5] - 0.3 * np.exp(-0.5 * 5.374445)) < 1e-15
    # H1(0) - O(1): d = (0.757 - 3, 0.586, 0): the same distance as O(0) - H2(1) by the mirror symmetry of the molecule
    assert abs(s[4, 0] - s[0, 5]) < 1e-16 and abs(h[4, 0] - h[0, 5]) < 1e-16
    # H1(0) - H1(1): both offsets cancel: r = 3;  H1(0) - H2(1): d = (0.757 + 0.757 - 3, 0, 0): r = 1.486
    assert abs(s[4, 4] - s[0, 0]) < 1e-16
    assert abs(s[4, 5] - 0.3 * np.exp(-0.5 * 1.486 ** 2)) < 1e-15
    assert abs(h[4, 5] - (-0.2 * np.exp(-1.486 / 1.5))) < 1e-15
    # block (1, 0) is the transpose of block (0, 1)
    h10, s10 = orc.two_centre_block(pos, box, 1, 0, m)
    assert np.array_equal(h10, h.T) and np.array_equal(s10, s.T)
    # on-site block: identity / orbital energies on the diagonal, zero between orbitals of one site,
    # O - H at r^2 = 0.757^2 + 0.586^2 = 0.916445, H1 - H2 at r = 1.514
    h00, s00 = orc.two_centre_block(pos, box, 0, 0, m)
    assert np.array_equal(np.diag(s00), np.ones(6)) and np.array_equal(np.diag(h00), [-1, -1, -1, -1, -0.5, -0.5])
    assert np.all(s00[:4, :4] == np.eye(4)) and np.all(h00[:4, :4] == -np.eye(4))
    assert abs(s00[0, 4] - 0.3 * np.exp(-0.5 * 0.916445)) < 1e-15 and abs(s00[3, 5] - s00[0, 4]) < 1e-16
    assert abs(h00[0, 4] - (-0.2 * np.exp(-np.sqrt(0.916445) / 1.5))) < 1e-15
    assert abs(s00[4, 5] - 0.3 * np.exp(-0.5 * 1.514 ** 2)) < 1e-15 and s00[4, 5] == s00[5, 4]
    # across the periodic boundary: centres 0 and 39 in a 40 A box are 1 A apart
    h02, s02 = orc.two_centre_block(pos, box, 0, 2, m)
    assert abs(s02[0, 0] - 0.3 * 0.6065306597126334) < 1e-15                   # 0.3 exp(-1/2)
    assert abs(h02[0, 0] - (-0.2 * 0.513417119032592)) < 1e-15                 # -0.2 exp(-1/1.5)


def test_generator_blocks_match_the_oracle_element_model(tiny_system):
    """nolsm_inputs.water._blocks (the shared input module) against the oracle's own, independently
    written two-centre model, every stored block of the tiny system and of a cutoff > L/2 system (per-site
    minimum image): equal to the last FP32 bit up to one ulp where exp() rounds differently."""
    m = _hand_model()
    assert gi.model_parameters(tiny_system)["site_offset"] == m["site_offset"]
    for system in (tiny_system, gi.make_water_system(32, 9.0)):
        worst = 0
        for i in range(0, system.n_mol, 3):
            for k in range(system.row_ptr[i], system.row_ptr[i + 1]):
                h, s = orc.two_centre_block(system.pos_q, system.box_q, i, int(system.col_idx[k]), m)
                for got, ref in ((system.h_val[k], h), (system.s_val[k], s)):
                    r32 = ref.astype(np.float32)
                    assert np.array_equal(got == 0, r32 == 0)
                    ulps = np.abs(got.view(np.int32).astype(np.int64) - r32.view(np.int32).astype(np.int64))
                    worst = max(worst, int(ulps.max()))
        assert worst <= 1, worst


def test_model_submatrix_equals_gathered_submatrix(tiny_system):
    """T_j evaluated from positions (model_submatrix) = T_j gathered from the block store (dense_submatrix),
    including the zero blocks of neighbour pairs that are themselves outside the cutoff."""
    s = tiny_system
    m = _hand_model()
    for j in (0, 7, 31):
        nbrs = s.col_idx[s.row_ptr[j]:s.row_ptr[j + 1]]
        hm, sm = orc.model_submatrix(s.pos_q, s.box_q, s.rc_q, nbrs, m)
        hg = orc.dense_submatrix(s.row_ptr, s.col_idx, s.h_val, nbrs)
        sg = orc.dense_submatrix(s.row_ptr, s.col_idx, s.s_val, nbrs)
        assert np.array_equal(hm == 0, hg == 0) and np.array_equal(sm == 0, sg == 0)
        assert (hm == 0).any()                                               # the pattern test is not vacuous
        assert np.abs(hm - hg).max() < 1e-7 and np.abs(sm - sg).max() < 1e-7  # FP32 rounding of the store


# ------------------------------------------------------------------ the acceptance evaluator itself
def test_sign_residual_pins():
    """||X^2 - I||_F / sqrt(n): diag(1.1, 1) -> sqrt(0.21^2) / sqrt(2) = 0.21 / sqrt(2); an exact
    involution -> 0; and the same quantity as newton_schulz_sign's residual history (computed there
    separately)."""
    assert abs(orc.sign_residual(np.diag([1.1, 1.0])) - 0.21 / np.sqrt(2.0)) < 1e-15
    assert abs(orc.sign_residual(np.diag([1.1, 1.0, 1.0, 1.0])) - 0.21 / 2.0) < 1e-15     # / sqrt(n), not / n
    refl = np.eye(5) - 2.0 * np.outer(np.ones(5), np.ones(5)) / 5.0
    assert orc.sign_residual(refl) < 1e-15
    a, q, lam = gi.make_gapped_symmetric(24, seed=3)
    a = a.astype(np.float64)
    x3, hist = orc.newton_schulz_sign(a, 4, scale=np.abs(lam).max(), history=True)
    x_k = a / np.abs(lam).max()
    for k in range(4):
        assert abs(orc.sign_residual(x_k) - hist[k]) < 1e-13
        x_k = orc.newton_schulz_sign(x_k, 1)


# ------------------------------------------------------------------ combination heuristic (row f3, Eq. 14)
def _csr(lists):
    rp = np.zeros(len(lists) + 1, dtype=np.int32)
    rp[1:] = np.cumsum([len(l) for l in lists])
    return rp, np.concatenate([np.asarray(l, dtype=np.int32) for l in lists])


def test_merge_criterion_eq14_hand_cases():
    """Eq. 14 on numbers worked by hand: identical sets always merge (n^3 < 2 n^3); disjoint sets
    never do ((a+b)^3 > a^3 + b^3); 10 and 10 rows with 8 common: 12^3 = 1728 < 2000 merges, with 7 common:
    13^3 = 2197 > 2000 does not; the threshold for equal sizes is n_common > (2 - 2^(1/3)) n = 0.74 n."""
    assert orc.merge_gain(5, 5, 5)
    assert not orc.merge_gain(4, 9, 0)
    assert orc.merge_gain(10, 10, 8) and not orc.merge_gain(10, 10, 7)
    assert orc.merge_gain(100, 100, 75) and not orc.merge_gain(100, 100, 74)
    # a small set inside a large one: 30^3 = 27000 < 27027 merges; one new row: 31^3 = 29791 > 27027 does not
    assert orc.merge_gain(30, 3, 3) and not orc.merge_gain(30, 3, 2)


def test_combination_heuristic_hand_built_examples():
    """Hand-built systems (lists include self, symmetric):
    (a) a clique of 4: every row set is {0,1,2,3}: everything merges into one cluster in the sweep d = 0;
    (b) two cliques {0,1,2} and {3,4,5} without a link: two clusters, no cross merge (disjoint sets never pay);
    (c) a chain 0-1-2-3-4 (each molecule sees its neighbours and itself): sets of size 2,3,3,3,2.  Sweep d = 0:
        cluster 1 absorbs 0 ({0,1} inside {0,1,2}: (3+2-2)^3 = 27 < 35), cluster 3 absorbs 4; sweep d = 1: cluster 1
        ({0,1,2}) looks at 2 ({1,2,3}): common 2, merged 4: 64 > 54, no; so three clusters remain: {0,1}, {2}, {3,4}."""
    rp, ci = _csr([[0, 1, 2, 3]] * 4)
    g = orc.combine_submatrices(rp, ci)
    assert g == [([0, 1, 2, 3], [0, 1, 2, 3])]
    rp, ci = _csr([[0, 1, 2]] * 3 + [[3, 4, 5]] * 3)
    assert orc.combine_submatrices(rp, ci) == [([0, 1, 2], [0, 1, 2]), ([3, 4, 5], [3, 4, 5])]
    rp, ci = _csr([[0, 1], [0, 1, 2], [1, 2, 3], [2, 3, 4], [3, 4]])
    assert orc.combine_submatrices(rp, ci) == [([0, 1], [0, 1, 2]), ([2], [1, 2, 3]), ([3, 4], [2, 3, 4])]


def test_combination_heuristic_invariants_on_water(tiny_system, tiny_solution):
    """On the generated system: the clusters partition the molecules, every owner's neighbour list lies inside its
    cluster's row set, the cubic work never exceeds the one-per-molecule value (each accepted merge lowers it by
    Eq. 14), and D from a combined submatrix equals the one-per-molecule D when the merged row set is the whole
    system (cutoff 9 A: every list is full, everything merges, the result is the full-matrix projector)."""
    s = tiny_system
    groups = orc.combine_submatrices(s.row_ptr, s.col_idx)
    owners = sorted(m for o, _ in groups for m in o)
    assert owners == list(range(s.n_mol))
    for o, r in groups:
        for j in o:
            assert set(s.col_idx[s.row_ptr[j]:s.row_ptr[j + 1]]) <= set(r)
    singles = [([j], list(s.col_idx[s.row_ptr[j]:s.row_ptr[j + 1]])) for j in range(s.n_mol)]
    assert orc.cubic_work(groups) <= orc.cubic_work(singles)
    assert len(groups) < s.n_mol                      # water-like lists overlap by ~ 0.8: merging pays
    full = gi.make_water_system(32, 9.0)
    g = orc.combine_submatrices(full.row_ptr, full.col_idx)
    assert len(g) == 1 and g[0][0] == list(range(32))
    sol = orc.solve_group(full.row_ptr, full.col_idx, full.h_val, full.s_val, *g[0])
    ref = orc.solve_system(full, mu=-0.85)
    for j in (0, 13, 31):
        cols = ref["solutions"][j].density_columns(-0.85)
        assert np.abs(sol.density_columns(j, -0.85) - cols).max() < 1e-12


def test_order3_sign_iteration_pins():
    """Scalar closed form (worked by hand): x = 0.5 -> e = 0.75 -> x (1 + 0.375 + 0.2109375) = 0.79296875; cubic
    convergence e' -> 5/8 e^3 (the first three terms of (1 - e)^(-1/2)); the fixed points are +-1; and the matrix
    iteration reaches Q sign(lam) Q^T (known by construction) in fewer iterations than Eq. 9."""
    assert orc.sign_iteration_order3(np.array([[0.5]]), 1)[0, 0] == 0.79296875
    x = np.array([[0.99]])
    e0 = 1 - 0.99 ** 2
    x1 = orc.sign_iteration_order3(x, 1)[0, 0]
    assert abs((1 - x1 * x1) / e0 ** 3 - 0.625) < 0.02
    assert orc.sign_iteration_order3(np.diag([1.0, -1.0]), 3).tolist() == [[1.0, 0.0], [0.0, -1.0]]
    a, q, lam = gi.make_gapped_symmetric(48, seed=7)
    a = a.astype(np.float64)
    sc = np.abs(lam).max()
    x3, r3 = orc.sign_iteration_order3(a, 8, scale=sc, history=True)
    x2, r2 = orc.newton_schulz_sign(a, 14, scale=sc, history=True)
    assert (r2 < 1e-2).any()
    assert np.abs(x3 - orc.sign_by_construction(q, lam)).max() < 1e-5      # FP32 input matrix
    assert np.argmax(r3 < 1e-2) < np.argmax(r2 < 1e-2)                     # fewer iterations to the same residual
