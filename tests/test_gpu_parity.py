"""Parity of the CUDA path (through the C ABI) with the FP64 oracle on the same seeded inputs.

Tolerances (BASELINE.json:north_star, restated in DESIGN.md "Tolerances"):
  neighbour lists / index sets   bit-exact
  gather                         bit-exact (it is a copy)
  D elements, max-abs            1e-5 (FP32 path)   5e-3 (FP16 operands / FP32 accumulate)
  ||X^2 - I||_F / sqrt(n)        <= 1e-2 (evaluated here in FP64 on the returned FP32 iterate)
  electron count                 |N_gpu - N_oracle| / n_mol <= 1e-3   (reading 16)
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL_D = {0: 5e-3, 1: 1e-5}      # keyed by precision: FP16_FP32 = 0, FP32 = 1
TOL_RESID = 1e-2
TOL_NE_PER_MOL = 1e-3
MU = -0.85                       # inside the gap of every generated system


@pytest.fixture(scope="module")
def nolsm():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2104_08245_b200 as m
    m.load_library()  # raises if libnolsm.so is missing: no fallback
    return m


@pytest.fixture(scope="module")
def torch_mod():
    import torch
    return torch


def _device_system(nolsm, system):
    H = nolsm.BlockSparse.from_numpy(system.row_ptr, system.col_idx, system.h_val)
    S = nolsm.BlockSparse(H.row_ptr, H.col_idx,
                          __import__("torch").as_tensor(system.s_val).contiguous().cuda())
    return H, S


@pytest.fixture(scope="module")
def mid_system():
    import nolsm_inputs as gi
    return gi.make_water_system(216, 8.0)


@pytest.fixture(scope="module")
def mid_solution(mid_system):
    import oracle.nolsm_oracle as orc
    return orc.solve_system(mid_system, mu=MU)


# ---------------------------------------------------------------------------------------------
# a0
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n_mol,cutoff", [(32, 6.0), (32, 9.0), (216, 8.0), (4096, 8.0)])
def test_neighbour_lists_bit_exact(nolsm, torch_mod, n_mol, cutoff):
    import nolsm_inputs as gi
    import oracle.nolsm_oracle as orc
    pos, box = gi.make_positions(n_mol)
    rc_q = int(round(cutoff * gi.GRID_PER_ANGSTROM))
    ctx = nolsm.Context()
    rp, ci = ctx.build_neighbours(torch_mod.as_tensor(pos).cuda(), box, rc_q)
    rp, ci = rp.cpu().numpy(), ci.cpu().numpy()
    if n_mol <= 216:
        rp_o, ci_o = orc.neighbour_list(pos, box, rc_q)
        assert np.array_equal(rp, rp_o) and np.array_equal(ci, ci_o)
    else:
        # oracle one molecule at a time on a sample + global invariants
        for j in [0, 1, 17, 2047, 4095]:
            assert np.array_equal(ci[rp[j]:rp[j + 1]], orc.neighbours_of(pos, box, rc_q, j))
        assert rp[0] == 0 and rp[-1] == ci.shape[0]
        rows = np.repeat(np.arange(n_mol), np.diff(rp))
        fwd = set(zip(rows.tolist(), ci.tolist()))
        assert all((c, r) in fwd for r, c in list(fwd)[:20000])  # symmetry on a sample
    ctx.close()


def test_neighbours_degenerate_cases(nolsm, torch_mod):
    ctx = nolsm.Context()
    # one molecule: its own neighbour; zero cutoff: self only
    pos = torch_mod.tensor([[5, 7, 9]], dtype=torch_mod.int32).cuda()
    rp, ci = ctx.build_neighbours(pos, [100, 100, 100], 10)
    assert rp.tolist() == [0, 1] and ci.tolist() == [0]
    pos = torch_mod.tensor([[0, 0, 0], [98, 0, 0], [50, 50, 50]], dtype=torch_mod.int32).cuda()
    rp, ci = ctx.build_neighbours(pos, [100, 100, 100], 0)
    assert rp.tolist() == [0, 1, 2, 3] and ci.tolist() == [0, 1, 2]
    # closed ball and the minimum image: |98-0| wraps to 2
    rp, ci = ctx.build_neighbours(pos, [100, 100, 100], 2)
    assert ci.tolist() == [0, 1, 0, 1, 2]
    rp, ci = ctx.build_neighbours(pos, [100, 100, 100], 1)
    assert ci.tolist() == [0, 1, 2]
    with pytest.raises(nolsm.NolsmError):
        ctx.build_neighbours(pos, [101, 100, 100], 1)  # odd box
    ctx.close()


# ---------------------------------------------------------------------------------------------
# a1
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("which", ["tiny", "mid"])
def test_gather_bitwise(nolsm, tiny_system, mid_system, which):
    import oracle.nolsm_oracle as orc
    system = tiny_system if which == "tiny" else mid_system
    H, S = _device_system(nolsm, system)
    ctx = nolsm.Context()
    count = system.n_mol if which == "tiny" else 24
    begin = 0 if which == "tiny" else 100
    batch = ctx.build_submatrices(H, S, begin, count)
    assert batch.size == count
    for local in ([0, 5, count - 1] if which == "mid" else range(count)):
        j = begin + local
        nbrs = system.col_idx[system.row_ptr[j]:system.row_ptr[j + 1]]
        for mat, val in ((nolsm.MAT_H, system.h_val), (nolsm.MAT_S, system.s_val)):
            ref = orc.dense_submatrix(system.row_ptr, system.col_idx, val, nbrs).astype(np.float32)
            got = batch.read(local, mat).cpu().numpy()
            assert got.shape == ref.shape
            assert np.array_equal(got.view(np.uint32), ref.view(np.uint32))
    empty = ctx.build_submatrices(H, S, 3, 0)
    assert empty.size == 0
    with pytest.raises(nolsm.NolsmError):
        ctx.build_submatrices(H, S, system.n_mol - 1, 2)
    ctx.close()


# ---------------------------------------------------------------------------------------------
# the GEMM building block
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kind,tol", [(0, 2e-5), (1, 2e-2), (2, 2e-5), (3, 2e-5)])
@pytest.mark.parametrize("n,batch", [(64, 3), (146, 5), (478, 2), (863, 2)])
def test_gemm_building_block(nolsm, torch_mod, kind, tol, n, batch):
    """C = A B and C = I - A B against FP64 numpy; kind 0 SIMT FP32, 1 tcgen05 FP16 operands,
    2 tcgen05 split-FP16, 3 tcgen05 half-split (A split, B exact in FP16: one stacked MMA per K step; its add-in
    goes through the staging buffers as a split FP16 pair with an FP32 result, the path of B1 = B0 + A0 R).
    Tolerances relative to sqrt(n) * max|A| * max|B| (rounding of a length-n
    dot product: FP32 ~ 6e-8 * sqrt(n); FP16 operands ~ 5e-4 * sqrt(n))."""
    rng = np.random.default_rng(n * 10 + kind)
    a = rng.uniform(-1, 1, (batch, n, n)).astype(np.float32)
    b = rng.uniform(-1, 1, (batch, n, n)).astype(np.float32)
    if kind == 3:
        b = b.astype(np.float16).astype(np.float32)
    cin = rng.uniform(-1, 1, (batch, n, n)).astype(np.float32)
    ref = a.astype(np.float64) @ b.astype(np.float64)
    scale = np.sqrt(n)
    ctx = nolsm.Context()
    ta, tb, tc = (torch_mod.as_tensor(x).cuda() for x in (a, b, cin))
    c, _ = ctx.gemm_batched(kind, ta, tb)
    err = np.abs(c.cpu().numpy() - ref).max() / scale
    assert err < tol, f"plain product: {err}"
    c, _ = ctx.gemm_batched(kind, ta, tb, cin=tc, alpha=0.5, beta=1.0)
    err = np.abs(c.cpu().numpy() - (0.5 * ref + cin)).max() / scale
    assert err < tol, f"axpby: {err}"
    c, r2 = ctx.gemm_batched(kind, ta, tb, ident=True)
    want = np.eye(n)[None] - ref
    err = np.abs(c.cpu().numpy() - want).max() / scale
    assert err < tol, f"identity-minus: {err}"
    r2_ref = (want ** 2).sum(axis=(1, 2))
    assert np.allclose(r2.cpu().numpy(), r2_ref, rtol=5e-3 if kind == 1 else 1e-4)
    ctx.close()


# ---------------------------------------------------------------------------------------------
# a2, a3: S^-1 and B = S^-1 H
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("which", ["tiny", "mid"])
@pytest.mark.parametrize("precision,tol", [(1, 2e-5), (0, 2e-4)])
def test_inverse_and_operator(nolsm, tiny_system, mid_system, precision, tol, which):
    """Eq. 15-17 converge to exactly S^-1: compare with LAPACK's inverse in FP64.
    The FP16 mode refines S^-1 to FP32 quality (reading 11), hence the tight bound there too.
    tiny: n ~ 146 (two tiles a side); mid: n ~ 478 (four tiles a side, several 64-row chunks per tile)."""
    import oracle.nolsm_oracle as orc
    system = tiny_system if which == "tiny" else mid_system
    begin, count = (0, system.n_mol) if which == "tiny" else (90, 20)
    H, S = _device_system(nolsm, system)
    ctx = nolsm.Context(nolsm.Config(precision=precision))
    batch = ctx.build_submatrices(H, S, begin, count)
    stats = ctx.sign_batched(batch, MU)
    assert stats.inv_iter_max > 0
    for local in ((0, 7, 31) if which == "tiny" else (0, 11, 19)):
        j = begin + local
        nbrs = system.col_idx[system.row_ptr[j]:system.row_ptr[j + 1]]
        s_sub = orc.dense_submatrix(system.row_ptr, system.col_idx, system.s_val, nbrs)
        h_sub = orc.dense_submatrix(system.row_ptr, system.col_idx, system.h_val, nbrs)
        sinv = np.linalg.inv(s_sub)
        got = batch.read(local, nolsm.MAT_SINV).cpu().numpy()
        assert np.abs(got - sinv).max() < tol
        got_b = batch.read(local, nolsm.MAT_B).cpu().numpy()
        assert np.abs(got_b - sinv @ h_sub).max() < 5 * tol
    ctx.close()


# ---------------------------------------------------------------------------------------------
# a4: sign iteration (dense microbench entry: sign known by construction)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision,tol_x", [(1, 2e-5), (0, 3e-3)])
@pytest.mark.parametrize("n,batch", [(256, 4), (200, 3), (512, 2)])
def test_sign_dense_against_construction(nolsm, torch_mod, precision, tol_x, n, batch):
    import nolsm_inputs as gi
    import oracle.nolsm_oracle as orc
    mats = [gi.make_gapped_symmetric(n, seed=7, index=i) for i in range(batch)]
    a = torch_mod.as_tensor(np.stack([m[0] for m in mats])).cuda()
    scale = torch_mod.as_tensor(np.array([np.abs(m[2]).max() for m in mats], dtype=np.float32)).cuda()
    ctx = nolsm.Context(nolsm.Config(precision=precision))
    x, stats = ctx.sign_dense_batched(a, scale)
    x = x.cpu().numpy()
    assert stats.n_unconverged == 0
    assert 6 <= stats.iter_min and stats.iter_max <= 14
    for i, (_, q, lam) in enumerate(mats):
        ref = orc.sign_by_construction(q, lam)
        assert np.abs(x[i] - ref).max() < tol_x
        assert orc.sign_residual(x[i]) <= TOL_RESID
    # fixed-iteration mode against the literal iteration of Eq. 9-10 in FP64
    k_fix = 5
    x5, st5 = ctx.sign_dense_batched(a, scale, fixed_iter=k_fix)
    assert st5.iter_min == k_fix and st5.iter_max == k_fix
    ref5 = orc.newton_schulz_sign(mats[0][0].astype(np.float64), k_fix, scale=float(np.abs(mats[0][2]).max()))
    assert np.abs(x5[0].cpu().numpy() - ref5).max() < (5e-3 if precision == 0 else 5e-5)
    # without a caller-supplied scale the norm bound is used: same limit
    x2, _ = ctx.sign_dense_batched(a, None)
    assert np.abs(x2[0].cpu().numpy() - orc.sign_by_construction(mats[0][1], mats[0][2])).max() < tol_x
    ctx.close()


def test_sign_degenerate_inputs(nolsm, torch_mod):
    ctx = nolsm.Context(nolsm.Config(precision=1))
    # 1x1 and diagonal matrices: sign is the sign of the entries
    a = torch_mod.tensor([[[0.3]], [[-0.7]]], dtype=torch_mod.float32).cuda()
    x, _ = ctx.sign_dense_batched(a, None)
    assert np.allclose(x.cpu().numpy().ravel(), [1.0, -1.0], atol=1e-5)
    d = np.diag(np.array([0.5, -0.25, 1.0, -1.0, 0.05], dtype=np.float32))[None]
    x, st = ctx.sign_dense_batched(torch_mod.as_tensor(d).cuda(), None)
    assert np.allclose(np.diag(x[0].cpu().numpy()), [1, -1, 1, -1, 1], atol=1e-5)
    # empty batch
    e = torch_mod.empty((0, 8, 8), dtype=torch_mod.float32).cuda()
    x, st = ctx.sign_dense_batched(e, None)
    assert x.shape[0] == 0
    # a singular matrix cannot converge: reported, not hidden
    z = torch_mod.zeros((1, 16, 16), dtype=torch_mod.float32).cuda()
    z[0, 0, 0] = 1.0
    x, st = ctx.sign_dense_batched(z, None, max_iter=8)
    assert st.n_unconverged == 1 and st.iter_max == 8
    ctx.close()


# ---------------------------------------------------------------------------------------------
# whole path, element by element
# ---------------------------------------------------------------------------------------------
def _check_density(nolsm, system, d_ref, mu, precision, ne_ref, mol_begin=0, mol_count=None):
    import torch
    H, S = _device_system(nolsm, system)
    D = S.like()
    ctx = nolsm.Context(nolsm.Config(precision=precision))
    mol_count = system.n_mol - mol_begin if mol_count is None else mol_count
    batch = ctx.build_submatrices(H, S, mol_begin, mol_count)
    stats = ctx.sign_batched(batch, mu)
    assert stats.n_unconverged == 0
    ne = torch.zeros(1, dtype=torch.float64, device="cuda")
    ne_diag = torch.zeros(1, dtype=torch.float64, device="cuda")
    q = torch.zeros(system.n_mol, dtype=torch.float64, device="cuda")
    ctx.scatter_density(batch, S, D, ne, q, ne_diag)
    lo, hi = system.row_ptr[mol_begin], system.row_ptr[mol_begin + mol_count]
    d = D.val.cpu().numpy()[lo:hi]
    err = np.abs(d - d_ref[lo:hi]).max()
    assert err < TOL_D[precision], f"max|dD| = {err}"
    # residual of the returned iterate, FP64, true n
    import oracle.nolsm_oracle as orc
    for local in (0, mol_count // 2, mol_count - 1):
        assert orc.sign_residual(batch.read(local, nolsm.MAT_X).cpu().numpy()) <= TOL_RESID
    # D is written only inside the pattern and only for the batch's molecules
    full = D.val.cpu().numpy()
    assert not full[:lo].any() and not full[hi:].any()
    ctx.close()
    return float(ne.item()), float(ne_diag.item()), q.cpu().numpy(), stats


@pytest.mark.parametrize("precision", [1, 0])
def test_density_tiny_all_molecules(nolsm, tiny_system, tiny_solution, precision):
    import oracle.nolsm_oracle as orc
    sols = tiny_solution["solutions"]
    d_ref = orc.density_blocks(sols, tiny_system.row_ptr, MU)
    ne_ref = orc.electron_count(sols, MU)
    ne, ne_diag, q, stats = _check_density(nolsm, tiny_system, d_ref, MU, precision, ne_ref)
    assert abs(ne - ne_ref) / tiny_system.n_mol <= TOL_NE_PER_MOL
    assert abs(ne_diag - ne_ref) / tiny_system.n_mol <= TOL_NE_PER_MOL
    q_ref = np.array([s.population(MU) for s in sols])
    worst = np.abs(q - q_ref).max()
    assert worst <= (2e-5 if precision == 1 else 5e-3), worst   # reading 16: reported per molecule
    # block contraction of the oracle on the GPU's D agrees with the GPU's own reduction
    assert stats.iter_max <= 14


@pytest.mark.parametrize("precision", [1, 0])
def test_density_mid_partial_batch(nolsm, mid_system, mid_solution, precision):
    """216 molecules, 8 A: n ~ 478 spans 4 row tiles with a ragged tail; a batch in the middle of the
    system checks mol_begin handling."""
    import oracle.nolsm_oracle as orc
    sols = mid_solution["solutions"]
    d_ref = orc.density_blocks(sols, mid_system.row_ptr, MU)
    begin, count = 50, 60
    ne_ref = sum(s.population(MU) for s in sols[begin:begin + count])
    ne, ne_diag, q, _ = _check_density(nolsm, mid_system, d_ref, MU, precision, ne_ref, begin, count)
    assert abs(ne - ne_ref) / count <= TOL_NE_PER_MOL
    assert abs(ne_diag - ne_ref) / count <= TOL_NE_PER_MOL


@pytest.mark.parametrize("precision", [1, 0])
def test_solve_mu_tiny(nolsm, tiny_system, tiny_solution, precision):
    """Bisection: mu is not unique (reading 14) -- parity is on D and N, and mu must
    lie on the oracle's plateau (max_j HOMO_j, min_j LUMO_j)."""
    import oracle.nolsm_oracle as orc
    sols = tiny_solution["solutions"]
    H, S = _device_system(nolsm, tiny_system)
    ctx = nolsm.Context(nolsm.Config(precision=precision))
    mu, ne, D, stats = ctx.solve_mu(H, S, tiny_system.n_electrons, -3.0, 0.0, tol_ne_per_mol=1e-3, max_steps=30)
    n_occ = {s.j: int((s.lam < tiny_solution["mu"]).sum()) for s in sols}
    homo, lumo = orc.mu_plateau(sols, lambda s: n_occ[s.j])
    assert homo < mu < lumo
    ne_ref = orc.electron_count(sols, mu)
    assert abs(ne - ne_ref) / tiny_system.n_mol <= TOL_NE_PER_MOL
    assert abs(ne - tiny_system.n_electrons) <= 1e-3 * tiny_system.n_mol
    d_ref = orc.density_blocks(sols, tiny_system.row_ptr, mu)
    assert np.abs(D.val.cpu().numpy() - d_ref).max() < TOL_D[precision]
    assert stats.mu_steps == tiny_solution["steps"]     # same midpoint sequence as the oracle's bisection
    assert abs(stats.ne_diag - ne_ref) / tiny_system.n_mol <= TOL_NE_PER_MOL
    # fixed number of evaluations (BASELINE configs[1]: "5 mu bisection steps"), bracket shrinks by 2^-4
    mu5, ne5, _, st5 = ctx.solve_mu(H, S, tiny_system.n_electrons, -3.0, 0.0, tol_ne_per_mol=-1.0, max_steps=5)
    assert st5.mu_steps == 5 and abs((st5.mu_hi - st5.mu_lo) - 3.0 / 16) < 1e-12
    # streaming through a small workspace gives the same D
    ctx2 = nolsm.Context(nolsm.Config(precision=precision, workspace_bytes=16 << 20))
    mu2, ne2, D2, st2 = ctx2.solve_mu(H, S, tiny_system.n_electrons, -3.0, 0.0, tol_ne_per_mol=1e-3, max_steps=30)
    assert st2.n_batches > 1 and mu2 == mu
    assert np.abs(D2.val.cpu().numpy() - D.val.cpu().numpy()).max() < TOL_D[precision]
    ctx.close()
    ctx2.close()


def test_single_evaluation_path_mid(nolsm, mid_system, mid_solution):
    """A single N(mu) evaluation (fixed chemical potential; max_steps = 1) takes the shortest form of
    the prepare stage in FP16 mode (reading 11): B is never written, X0 = (B0 + A0 R - mu I)/s_j comes out
    of the last product's epilogue.  Same D, N and populations as the oracle, the same iteration counts as the
    path that forms B (max_steps = 2 evaluates the same mu first), and D within rounding of that path."""
    import oracle.nolsm_oracle as orc
    sols = mid_solution["solutions"]
    H, S = _device_system(nolsm, mid_system)
    ctx = nolsm.Context(nolsm.Config(precision=0))
    lo, hi = MU - 0.1, MU + 0.1
    mu1, ne1, D1, st1 = ctx.solve_mu(H, S, mid_system.n_electrons, lo, hi, tol_ne_per_mol=-1.0, max_steps=1)
    assert mu1 == MU
    d_ref = orc.density_blocks(sols, mid_system.row_ptr, MU)
    assert np.abs(D1.val.cpu().numpy() - d_ref).max() < TOL_D[0]
    ne_ref = orc.electron_count(sols, MU)
    assert abs(ne1 - ne_ref) / mid_system.n_mol <= TOL_NE_PER_MOL
    # the general path: tolerance met at the first midpoint, but a second step was allowed, so B was formed
    mu2, ne2, D2, st2 = ctx.solve_mu(H, S, mid_system.n_electrons, lo, hi, tol_ne_per_mol=1.0, max_steps=2)
    assert mu2 == MU and st2.mu_steps == 1
    assert (st1.last.iter_min, st1.last.iter_max) == (st2.last.iter_min, st2.last.iter_max)
    # two FP16-mode evaluations with different scales s_j: each is ~2e-4 from the oracle (bound 5e-3)
    assert np.abs(D1.val.cpu().numpy() - D2.val.cpu().numpy()).max() < 6e-4
    assert abs(ne1 - ne2) / mid_system.n_mol < 2e-4
    ctx.close()


@pytest.mark.parametrize("which", ["tiny", "mid"])
def test_a_priori_stop_of_the_inverse_iteration(nolsm, tiny_system, mid_system, which):
    """Eq. 15-17, FP16 mode (reading 11): from ||E_k||_1 the next residual is bounded before iteration k is
    finished (E_{k+1} = 3/4 E_k^2 + 1/4 E_k^3; pinned on the oracle in test_oracle_pins.py); when the bound passes,
    only Z_{k+1} is formed.  NOLSM_FLAG_NO_PREDICT decides every stop on a measured residual instead: it forms
    Y_{k+1} and E_{k+1} as well and then takes the SAME Z_{k+1} -- so D must be bitwise equal and the product count
    two per submatrix higher."""
    system = tiny_system if which == "tiny" else mid_system
    H, S = _device_system(nolsm, system)
    out = {}
    for flags in (0, nolsm.FLAG_NO_PREDICT):
        ctx = nolsm.Context(nolsm.Config(precision=0, flags=flags))
        mu, ne, D, st = ctx.solve_mu(H, S, system.n_electrons, MU - 0.1, MU + 0.1, tol_ne_per_mol=-1.0, max_steps=1)
        out[flags] = (D.val.cpu().numpy().copy(), ne, st.last.gemms, st.last.inv_iter_max)
        ctx.close()
    ahead, measured = out[0], out[nolsm.FLAG_NO_PREDICT]
    assert np.array_equal(ahead[0].view(np.uint32), measured[0].view(np.uint32))
    assert abs(ahead[1] - measured[1]) <= 1e-9 * abs(measured[1])   # same D; the trace is summed with atomics
    assert ahead[3] == measured[3]                                  # same number of Z updates
    assert measured[2] - ahead[2] == 2 * system.n_mol               # Y_{k+1} and E_{k+1} were never formed


def test_fp32_whole_path_two_refinements(nolsm, mid_system, mid_solution):
    """FP32 mode of nolsm_solve_mu (reading 11): Eq. 15-17 runs on FP16 operands to the a-priori stop, then
    B and the own columns of S^-1 are refined twice with their residuals on split operands (errors F^3 B, F^3 V with
    ||F||_2 <= 1e-2; pinned on the oracle in test_oracle_pins.py).  D, N and the populations against the oracle at the
    FP32 tolerances, and against the path that iterates Eq. 15-17 itself on split operands (NOLSM_FLAG_NO_PREDICT)."""
    import oracle.nolsm_oracle as orc
    import torch
    sols = mid_solution["solutions"]
    H, S = _device_system(nolsm, mid_system)
    d_ref = orc.density_blocks(sols, mid_system.row_ptr, MU)
    ne_ref = orc.electron_count(sols, MU)
    out = {}
    for flags in (0, nolsm.FLAG_NO_PREDICT):
        ctx = nolsm.Context(nolsm.Config(precision=1, flags=flags))
        q = torch.zeros(mid_system.n_mol, dtype=torch.float64, device="cuda")
        mu, ne, D, st = ctx.solve_mu(H, S, mid_system.n_electrons, MU - 0.1, MU + 0.1, tol_ne_per_mol=-1.0,
                                     max_steps=1, q_mol=q)
        d = D.val.cpu().numpy().copy()
        assert np.abs(d - d_ref).max() < TOL_D[1]
        assert abs(ne - ne_ref) / mid_system.n_mol <= TOL_NE_PER_MOL
        pop = np.array([s.population(MU) for s in sols])
        assert np.abs(q.cpu().numpy() - pop).max() < 2e-5
        out[flags] = (d, st.last.gemms, st.last.inv_iter_max)
        ctx.close()
    fast, slow = out[0], out[nolsm.FLAG_NO_PREDICT]
    assert np.abs(fast[0] - slow[0]).max() < 5e-6
    assert fast[1] < slow[1] and fast[2] < slow[2]      # fewer products, fewer iterations of Eq. 15-17


@pytest.mark.parametrize("which", ["tiny", "mid"])
def test_lowdin_form(nolsm, tiny_system, tiny_solution, mid_system, mid_solution, which):
    """SURVEY 8(f)#4, NOLSM_FLAG_LOWDIN: sign of the SYMMETRIC S^-1/2 H S^-1/2 - mu I with S^-1/2 from Eq. 15-17, and
    D[:, own] = Z (1/2 (I - X~)) Z[:, own] / s as thin products.  Same D, N and populations as the oracle (whose Loewdin
    restatement is pinned against the generalized eigenproblem in test_oracle_pins.py) at the FP32 tolerances; the
    flag is refused in FP16 mode."""
    import oracle.nolsm_oracle as orc
    import torch
    system, solution = (tiny_system, tiny_solution) if which == "tiny" else (mid_system, mid_solution)
    sols = solution["solutions"]
    H, S = _device_system(nolsm, system)
    ctx = nolsm.Context(nolsm.Config(precision=1, flags=nolsm.FLAG_LOWDIN))
    q = torch.zeros(system.n_mol, dtype=torch.float64, device="cuda")
    mu, ne, D, st = ctx.solve_mu(H, S, system.n_electrons, MU - 0.1, MU + 0.1, tol_ne_per_mol=-1.0, max_steps=1,
                                 q_mol=q)
    assert mu == MU
    d_ref = orc.density_blocks(sols, system.row_ptr, MU)
    assert np.abs(D.val.cpu().numpy() - d_ref).max() < TOL_D[1]
    assert abs(ne - orc.electron_count(sols, MU)) / system.n_mol <= TOL_NE_PER_MOL
    pop = np.array([s.population(MU) for s in sols])
    assert np.abs(q.cpu().numpy() - pop).max() < 2e-5
    assert st.last.n_unconverged == 0
    # a second evaluation on the same context (bisection step with resident batches) and the streaming path
    mu2, ne2, D2, st2 = ctx.solve_mu(H, S, system.n_electrons, MU - 0.3, MU + 0.1, tol_ne_per_mol=-1.0, max_steps=2)
    d_ref2 = orc.density_blocks(sols, system.row_ptr, mu2)
    assert np.abs(D2.val.cpu().numpy() - d_ref2).max() < TOL_D[1]
    ctx.close()
    ctx16 = nolsm.Context(nolsm.Config(precision=0, flags=nolsm.FLAG_LOWDIN))
    with pytest.raises(nolsm.NolsmError, match="LOWDIN"):
        ctx16.solve_mu(H, S, system.n_electrons, MU - 0.1, MU + 0.1, max_steps=1)
    ctx16.close()


def test_rescaled_first_sign_iteration(nolsm, mid_system, mid_solution):
    """DESIGN.md reading 5: the first product of the sign iteration (X0^2) also gives ||X0^2||_1 >= rho(X0)^2, and
    iteration 0 is applied to a X0, a = 1.7 / sqrt(||X0^2||_1) in [1, 1.7] (oracle: newton_schulz_sign_rescaled, pinned in
    test_oracle_pins.py).  Same D and N as the oracle with and without it (NOLSM_FLAG_NO_RESCALE), never more iterations,
    and the result is bitwise reproducible although the norm is gathered with atomics (integer sums)."""
    import oracle.nolsm_oracle as orc
    sols = mid_solution["solutions"]
    H, S = _device_system(nolsm, mid_system)
    d_ref = orc.density_blocks(sols, mid_system.row_ptr, MU)
    ne_ref = orc.electron_count(sols, MU)
    out = {}
    for flags in (0, nolsm.FLAG_NO_RESCALE):
        ctx = nolsm.Context(nolsm.Config(precision=0, flags=flags))
        runs = []
        for rep in range(2):
            mu, ne, D, st = ctx.solve_mu(H, S, mid_system.n_electrons, MU - 0.1, MU + 0.1, tol_ne_per_mol=-1.0,
                                         max_steps=1)
            runs.append(D.val.cpu().numpy().copy())
        assert np.array_equal(runs[0].view(np.uint32), runs[1].view(np.uint32))
        assert np.abs(runs[0] - d_ref).max() < TOL_D[0]
        assert abs(ne - ne_ref) / mid_system.n_mol <= TOL_NE_PER_MOL
        assert st.last.n_unconverged == 0 and st.last.worst_residual <= TOL_RESID
        out[flags] = (st.last.iter_min, st.last.iter_max, st.last.iter_sum)
        ctx.close()
    assert out[0][1] <= out[nolsm.FLAG_NO_RESCALE][1] and out[0][2] < out[nolsm.FLAG_NO_RESCALE][2]
    # the user-level entry point takes the same path: X against the oracle's sign function of the submatrix
    ctx = nolsm.Context(nolsm.Config(precision=0))
    batch = ctx.build_submatrices(H, S, 100, 4)
    st = ctx.sign_batched(batch, MU)
    x = batch.read(1, nolsm.MAT_X).cpu().numpy().astype(np.float64)
    sol = sols[101]
    sign_ref = np.eye(len(sol.s_sub)) - 2.0 * sol.density(MU) @ sol.s_sub
    assert np.abs(x - sign_ref).max() < 2e-3 and orc.sign_residual(x) <= TOL_RESID
    ctx.close()


# ---------------------------------------------------------------------------------------------
# BASELINE sizes, sampled (the oracle solves the sampled molecules one by one)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name,precision,begin,count,sample", [
    ("w4096", 1, 1000, 296, [0, 150, 295]),
    ("w4096", 0, 2000, 296, [1, 100, 294]),
    ("w32768", 0, 20000, 148, [0, 147]),
])
def test_baseline_configs_sampled(nolsm, name, precision, begin, count, sample):
    import torch
    import nolsm_inputs as gi
    import oracle.nolsm_oracle as orc
    n_mol, cutoff = gi.CONFIGS[name]
    system = gi.make_water_system(n_mol, cutoff)
    H, S = _device_system(nolsm, system)
    D = S.like()
    ctx = nolsm.Context(nolsm.Config(precision=precision))
    batch = ctx.build_submatrices(H, S, begin, count)
    stats = ctx.sign_batched(batch, MU)
    assert stats.n_unconverged == 0
    ne = torch.zeros(1, dtype=torch.float64, device="cuda")
    q = torch.zeros(n_mol, dtype=torch.float64, device="cuda")
    ctx.scatter_density(batch, S, D, ne, q, None)
    d = D.val.cpu().numpy()
    q = q.cpu().numpy()
    for local in sample:
        j = begin + local
        sol = orc.solve_molecule(system.row_ptr, system.col_idx, system.h_val, system.s_val, j)
        ref = sol.density_columns(MU).reshape(-1, 6, 6)
        lo = system.row_ptr[j]
        err = np.abs(d[lo:lo + ref.shape[0]] - ref).max()
        assert err < TOL_D[precision], f"molecule {j}: max|dD| = {err}"
        assert abs(q[j] - sol.population(MU)) < (2e-5 if precision == 1 else 5e-3)
        assert orc.sign_residual(batch.read(local, nolsm.MAT_X).cpu().numpy()) <= TOL_RESID
    # property that holds at any size: every molecule carries ~8 electrons (plateau, reading 14)
    qs = q[begin:begin + count]
    assert np.abs(qs - 8.0).max() < 0.03
    assert abs(ne.item() - qs.sum()) < 1e-6 * count
    ctx.close()


# ---------------------------------------------------------------------------------------------
# the optional pair engines (cta_group::2 pair tiles / cluster multicast of the B operand)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("flag", ["FLAG_PAIR", "FLAG_SINGLE"])
@pytest.mark.parametrize("precision", [0, 1])
def test_pair_engines_density_tiny_and_mid(nolsm, tiny_system, tiny_solution, mid_system, mid_solution, flag, precision):
    """Same parity bounds as the default engine, through nolsm_solve_mu (tiny) and a partial batch (mid:
    n ~ 478 = 4 row tiles, so the 256-row pair tiles have a ragged second half)."""
    import torch
    import oracle.nolsm_oracle as orc
    flags = getattr(nolsm, flag)
    sols = tiny_solution["solutions"]
    H, S = _device_system(nolsm, tiny_system)
    ctx = nolsm.Context(nolsm.Config(precision=precision, flags=flags))
    mu, ne, D, stats = ctx.solve_mu(H, S, tiny_system.n_electrons, -3.0, 0.0, tol_ne_per_mol=1e-3, max_steps=30)
    d_ref = orc.density_blocks(sols, tiny_system.row_ptr, mu)
    assert np.abs(D.val.cpu().numpy() - d_ref).max() < TOL_D[precision]
    assert abs(ne - orc.electron_count(sols, mu)) / tiny_system.n_mol <= TOL_NE_PER_MOL
    ctx.close()
    # mid system, molecules 50..109
    sols = mid_solution["solutions"]
    d_ref = orc.density_blocks(sols, mid_system.row_ptr, MU)
    H, S = _device_system(nolsm, mid_system)
    D = S.like()
    ctx = nolsm.Context(nolsm.Config(precision=precision, flags=flags))
    batch = ctx.build_submatrices(H, S, 50, 60)
    st = ctx.sign_batched(batch, MU)
    assert st.n_unconverged == 0
    ne_t = torch.zeros(1, dtype=torch.float64, device="cuda")
    ctx.scatter_density(batch, S, D, ne_t, None, None)
    lo, hi = mid_system.row_ptr[50], mid_system.row_ptr[110]
    assert np.abs(D.val.cpu().numpy()[lo:hi] - d_ref[lo:hi]).max() < TOL_D[precision]
    ctx.close()


@pytest.mark.parametrize("flag", ["FLAG_PAIR", "FLAG_SINGLE"])
@pytest.mark.parametrize("kind,tol", [(1, 2e-2), (2, 2e-5), (3, 2e-5)])
@pytest.mark.parametrize("n,batch", [(64, 3), (146, 5), (300, 2), (863, 2)])
def test_pair_engines_building_block(nolsm, torch_mod, flag, kind, tol, n, batch):
    rng = np.random.default_rng(n * 7 + kind)
    a = rng.uniform(-1, 1, (batch, n, n)).astype(np.float32)
    b = rng.uniform(-1, 1, (batch, n, n)).astype(np.float32)
    if kind == 3:   # half-split: the pair kernel runs it as two MMAs per K step, the single-CTA one as one stacked MMA
        b = b.astype(np.float16).astype(np.float32)
    cin = rng.uniform(-1, 1, (batch, n, n)).astype(np.float32)
    ref = a.astype(np.float64) @ b.astype(np.float64)
    ctx = nolsm.Context(nolsm.Config(flags=getattr(nolsm, flag)))
    ta, tb, tc = (torch_mod.as_tensor(x).cuda() for x in (a, b, cin))
    c, _ = ctx.gemm_batched(kind, ta, tb, cin=tc, alpha=0.5, beta=1.0)
    assert np.abs(c.cpu().numpy() - (0.5 * ref + cin)).max() / np.sqrt(n) < tol
    c, r2 = ctx.gemm_batched(kind, ta, tb, ident=True)
    want = np.eye(n)[None] - ref
    assert np.abs(c.cpu().numpy() - want).max() / np.sqrt(n) < tol
    assert np.allclose(r2.cpu().numpy(), (want ** 2).sum(axis=(1, 2)), rtol=5e-3 if kind == 1 else 1e-4)
    ctx.close()


# ---------------------------------------------------------------------------------------------
# energy-weighted density and electronic energy (Eq. 7, 8, 11, 13)
# ---------------------------------------------------------------------------------------------
TOL_W = {0: 5e-3, 1: 2e-5}       # |W| <~ 2.5 |D| (H0 eigenvalues down to -2.5 Ha): same relative bound as D
TOL_E_PER_MOL = {0: 2e-3, 1: 2e-5}


@pytest.mark.parametrize("precision", [1, 0])
def test_energy_weighted_density_tiny(nolsm, tiny_system, tiny_solution, precision):
    import oracle.nolsm_oracle as orc
    sols = tiny_solution["solutions"]
    H, S = _device_system(nolsm, tiny_system)
    ctx = nolsm.Context(nolsm.Config(precision=precision))
    ne, e, D, W, stats = ctx.evaluate(H, S, MU)
    d_ref = orc.density_blocks(sols, tiny_system.row_ptr, MU)
    w_ref = orc.energy_weighted_blocks(sols, tiny_system.row_ptr, MU)
    assert np.abs(D.val.cpu().numpy() - d_ref).max() < TOL_D[precision]
    assert np.abs(W.val.cpu().numpy() - w_ref).max() < TOL_W[precision]
    e_ref = orc.electronic_energy_blocks(tiny_system.row_ptr, tiny_system.col_idx, d_ref, tiny_system.h_val)
    assert abs(e - e_ref) / tiny_system.n_mol < TOL_E_PER_MOL[precision]
    # the GPU's own reduction agrees with the oracle's contraction of the GPU's D
    e_own = orc.electronic_energy_blocks(tiny_system.row_ptr, tiny_system.col_idx, D.val.cpu().numpy(), tiny_system.h_val)
    assert abs(e - e_own) < 1e-4
    assert abs(ne - orc.electron_count(sols, MU)) / tiny_system.n_mol <= TOL_NE_PER_MOL
    # E only (no W store)
    ne2, e2, _, W2, _ = ctx.evaluate(H, S, MU, want_w=False)
    assert W2 is None and abs(e2 - e) < 1e-6
    ctx.close()


@pytest.mark.parametrize("precision", [1, 0])
def test_energy_weighted_density_mid_batch(nolsm, mid_system, mid_solution, precision):
    """Batch-level entry on a partial batch (n ~ 478): W columns and the batch's share of Tr(D H0)."""
    import torch
    import oracle.nolsm_oracle as orc
    sols = mid_solution["solutions"]
    begin, count = 50, 60
    H, S = _device_system(nolsm, mid_system)
    D, W = S.like(), S.like()
    ctx = nolsm.Context(nolsm.Config(precision=precision))
    batch = ctx.build_submatrices(H, S, begin, count)
    ctx.sign_batched(batch, MU)
    ne = torch.zeros(1, dtype=torch.float64, device="cuda")
    e = torch.zeros(1, dtype=torch.float64, device="cuda")
    ctx.scatter_density(batch, S, D, ne, None, None)
    ctx.scatter_energy(batch, H, D, W, e)
    lo, hi = mid_system.row_ptr[begin], mid_system.row_ptr[begin + count]
    w_ref = orc.energy_weighted_blocks(sols[begin:begin + count], mid_system.row_ptr, MU)
    d_ref = orc.density_blocks(sols[begin:begin + count], mid_system.row_ptr, MU)
    w = W.val.cpu().numpy()
    assert np.abs(w[lo:hi] - w_ref[lo:hi]).max() < TOL_W[precision]
    assert not w[:lo].any() and not w[hi:].any()
    e_ref = float(np.einsum("kop,kpo->", d_ref[lo:hi], mid_system.h_val[lo:hi].astype(np.float64)))
    assert abs(e.item() - e_ref) / count < TOL_E_PER_MOL[precision]
    ctx.close()


# ---------------------------------------------------------------------------------------------
# more shapes: isolated molecules (n = 6), config-4-sized submatrices (n ~ 1489), larger microbench
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision", [1, 0])
def test_isolated_molecules_n6(nolsm, precision):
    """Cutoff 1 A: every neighbour list is the molecule itself, every submatrix is 6 x 6 (one padded tile)."""
    import nolsm_inputs as gi
    import oracle.nolsm_oracle as orc
    system = gi.make_water_system(32, 1.0)
    assert system.nnzb == 32
    sol = orc.solve_system(system, mu=MU)
    H, S = _device_system(nolsm, system)
    ctx = nolsm.Context(nolsm.Config(precision=precision))
    ne, e, D, W, stats = ctx.evaluate(H, S, MU)
    d_ref = orc.density_blocks(sol["solutions"], system.row_ptr, MU)
    w_ref = orc.energy_weighted_blocks(sol["solutions"], system.row_ptr, MU)
    assert np.abs(D.val.cpu().numpy() - d_ref).max() < TOL_D[precision]
    assert np.abs(W.val.cpu().numpy() - w_ref).max() < TOL_W[precision]
    assert abs(ne - orc.electron_count(sol["solutions"], MU)) / 32 <= TOL_NE_PER_MOL
    ctx.close()


def test_config4_sized_submatrices_sampled(nolsm):
    """4096 molecules at the 12 A cutoff of BASELINE configs[3]: n ~ 1489 (12 row tiles, 6 column tiles)."""
    import torch
    import nolsm_inputs as gi
    import oracle.nolsm_oracle as orc
    system = gi.make_water_system(4096, 12.0)
    H, S = _device_system(nolsm, system)
    D = S.like()
    ctx = nolsm.Context(nolsm.Config(precision=0))
    begin, count = 2100, 40
    batch = ctx.build_submatrices(H, S, begin, count)
    stats = ctx.sign_batched(batch, MU)
    assert stats.n_unconverged == 0
    ne = torch.zeros(1, dtype=torch.float64, device="cuda")
    q = torch.zeros(system.n_mol, dtype=torch.float64, device="cuda")
    ctx.scatter_density(batch, S, D, ne, q, None)
    d = D.val.cpu().numpy()
    for local in (0, 39):
        j = begin + local
        sol = orc.solve_molecule(system.row_ptr, system.col_idx, system.h_val, system.s_val, j)
        assert sol.n > 1400
        ref = sol.density_columns(MU).reshape(-1, 6, 6)
        lo = system.row_ptr[j]
        assert np.abs(d[lo:lo + ref.shape[0]] - ref).max() < TOL_D[0]
        assert abs(q[j].item() - sol.population(MU)) < 5e-3
        assert orc.sign_residual(batch.read(local, nolsm.MAT_X).cpu().numpy()) <= TOL_RESID
    ctx.close()


@pytest.mark.parametrize("precision,tol_x", [(1, 2e-5), (0, 3e-3)])
def test_sign_dense_n1024(nolsm, torch_mod, precision, tol_x):
    import nolsm_inputs as gi
    import oracle.nolsm_oracle as orc
    mats = [gi.make_gapped_symmetric(1024, seed=11, index=i) for i in range(2)]
    a = torch_mod.as_tensor(np.stack([m[0] for m in mats])).cuda()
    scale = torch_mod.as_tensor(np.array([np.abs(m[2]).max() for m in mats], dtype=np.float32)).cuda()
    ctx = nolsm.Context(nolsm.Config(precision=precision))
    x, stats = ctx.sign_dense_batched(a, scale)
    assert stats.n_unconverged == 0
    for i, (_, q, lam) in enumerate(mats):
        assert np.abs(x[i].cpu().numpy() - orc.sign_by_construction(q, lam)).max() < tol_x
    ctx.close()


def test_w32768_whole_step_in_bench_configuration_sampled(nolsm):
    """BASELINE configs[2] at full size through the call bench.py times (nolsm_solve_mu, 24 GiB workspace,
    38 streamed batches, default engine): sampled molecules against the oracle, plus properties that hold
    for every molecule (plateau populations, pattern-only writes)."""
    import torch
    import nolsm_inputs as gi
    import oracle.nolsm_oracle as orc
    n_mol, cutoff = gi.CONFIGS["w32768"]
    system = gi.make_water_system(n_mol, cutoff)
    H, S = _device_system(nolsm, system)
    ctx = nolsm.Context(nolsm.Config(precision=0, workspace_bytes=24 << 30))
    q = torch.zeros(n_mol, dtype=torch.float64, device="cuda")
    mu, ne, D, stats = ctx.solve_mu(H, S, system.n_electrons, 2 * MU, 0.0, tol_ne_per_mol=-1.0, max_steps=1, q_mol=q)
    assert mu == MU and stats.n_batches > 30 and stats.last.n_unconverged == 0
    assert 8 <= stats.last.iter_min and stats.last.iter_max <= 12
    d = D.val.cpu().numpy()
    qh = q.cpu().numpy()
    # first / last batch and fourteen spread in between
    for j in (0, 1, 700, 2047, 4096, 8191, 12345, 16384, 20000, 22222, 24576, 28000, 30000, 32000, 32766, 32767):
        sol = orc.solve_molecule(system.row_ptr, system.col_idx, system.h_val, system.s_val, j)
        ref = sol.density_columns(MU).reshape(-1, 6, 6)
        lo = system.row_ptr[j]
        assert np.abs(d[lo:lo + ref.shape[0]] - ref).max() < TOL_D[0], j
        assert abs(qh[j] - sol.population(MU)) < 5e-3
    # a0 at this size: sixteen sampled rows of the device-built neighbour list, bit-exact against the oracle
    pos = torch.as_tensor(system.pos_q).cuda()
    rp, ci = ctx.build_neighbours(pos, system.box_q, system.rc_q, cap=system.nnzb)
    rp_h, ci_h = rp.cpu().numpy(), ci.cpu().numpy()
    assert np.array_equal(rp_h, system.row_ptr)
    for j in range(5, n_mol, n_mol // 16):
        assert np.array_equal(ci_h[rp_h[j]:rp_h[j + 1]], orc.neighbours_of(system.pos_q, system.box_q, system.rc_q, j))
    assert np.abs(qh - 8.0).max() < 0.03          # every molecule sits on the plateau (reading 14)
    assert abs(ne - qh.sum()) < 1e-6 * n_mol
    assert abs(ne - system.n_electrons) / n_mol < 1e-3
    assert np.isfinite(d).all()
    ctx.close()


@pytest.mark.parametrize("flag", [0, "FLAG_PAIR", "FLAG_SINGLE"])
def test_run_to_run_bitwise_identical(nolsm, flag):
    """The tile schedule is dynamic (claim order and timing differ from run to run) but every tile's arithmetic
    is fixed, so two runs must give bit-identical D: any race in the dependency protocol (a tile reading an
    operand before its producer finished) would show up here."""
    import torch
    import nolsm_inputs as gi
    system = gi.make_water_system(*gi.CONFIGS["w4096"])
    H, S = _device_system(nolsm, system)
    flags = getattr(nolsm, flag) if flag else 0
    runs = []
    for _ in range(2):
        ctx = nolsm.Context(nolsm.Config(precision=0, flags=flags))
        mu, ne, D, st = ctx.solve_mu(H, S, system.n_electrons, 2 * MU, 0.0, tol_ne_per_mol=-1.0, max_steps=1)
        runs.append((D.val.clone(), ne))
        ctx.close()
    assert torch.equal(runs[0][0], runs[1][0])
    assert abs(runs[0][1] - runs[1][1]) < 1e-6


# ---------------------------------------------------------------------------------------------
# a1': elements evaluated on the device from the positions instead of gathered
# ---------------------------------------------------------------------------------------------
def _attach_model(nolsm, ctx, system, eval_fp32=False):
    import torch
    import nolsm_inputs as gi
    pos = torch.as_tensor(system.pos_q).contiguous().cuda()
    ctx.set_model(pos, eval_fp32=eval_fp32, **gi.model_parameters(system))
    return pos


@pytest.mark.parametrize("which", ["tiny", "tiny9", "mid"])
def test_generated_submatrices_match_block_store(nolsm, tiny_system, mid_system, which):
    """Same T_j(H), T_j(S) as the oracle's own two-centre model evaluated from the positions
    (oracle.model_submatrix, pinned on hand values in test_oracle_pins.py), and as the oracle's gather of the
    generator's blocks.  All sides evaluate the model in FP64 in the same operation order and round once to FP32,
    so the only admissible difference is exp()'s last FP64 bit crossing an FP32 rounding boundary: at most one
    FP32 ulp, on at most 1e-5 of the elements.
    tiny9 (cutoff 9 A > half the 9.86 A box) exercises the per-site minimum image."""
    import oracle.nolsm_oracle as orc
    import nolsm_inputs as gi
    system = {"tiny": tiny_system, "mid": mid_system}.get(which) or gi.make_water_system(32, 9.0)
    H, S = _device_system(nolsm, system)
    zeros = nolsm.BlockSparse(H.row_ptr, H.col_idx, H.val * 0)   # the stores must not be read
    ctx = nolsm.Context()
    _attach_model(nolsm, ctx, system)
    count = 24 if which == "mid" else system.n_mol
    begin = 100 if which == "mid" else 0
    batch = ctx.build_submatrices(zeros, zeros, begin, count)
    n_elem = n_diff = 0
    model = gi.model_parameters(system)
    for local in ([0, 5, count - 1] if which == "mid" else range(0, count, 4)):
        j = begin + local
        nbrs = system.col_idx[system.row_ptr[j]:system.row_ptr[j + 1]]
        h_model, s_model = orc.model_submatrix(system.pos_q, system.box_q, system.rc_q, nbrs, model)
        for mat, val, from_model in ((nolsm.MAT_H, system.h_val, h_model), (nolsm.MAT_S, system.s_val, s_model)):
            got = batch.read(local, mat).cpu().numpy()
            for ref in (from_model.astype(np.float32),
                        orc.dense_submatrix(system.row_ptr, system.col_idx, val, nbrs).astype(np.float32)):
                assert got.shape == ref.shape
                assert np.array_equal(got == 0, ref == 0)              # the pattern is integer work: exact
                ulp = np.spacing(np.abs(ref))
                assert (np.abs(got - ref) <= ulp).all()
                n_elem += ref.size
                n_diff += int((got.view(np.uint32) != ref.view(np.uint32)).sum())
    assert n_diff <= max(2, int(1e-5 * n_elem)), (n_diff, n_elem)
    ctx.set_model(None)                                            # detached: gathers again
    batch = ctx.build_submatrices(H, S, begin, 1)
    ref = orc.dense_submatrix(system.row_ptr, system.col_idx, system.h_val,
                              system.col_idx[system.row_ptr[begin]:system.row_ptr[begin + 1]]).astype(np.float32)
    assert np.array_equal(batch.read(0, nolsm.MAT_H).cpu().numpy(), ref)
    ctx.close()


@pytest.mark.parametrize("which", ["tiny9", "mid"])
def test_generated_submatrices_fp32_sfu(nolsm, mid_system, which):
    """The paper's own flavour (FP32 arithmetic, SFU exponentials): same zero pattern, elements
    within 1e-6 of the FP64 evaluation (|S|, |H| <= 1; __expf is good to 2^-21 relative, r^2 to 1e-6 A^2)."""
    import oracle.nolsm_oracle as orc
    import nolsm_inputs as gi
    system = mid_system if which == "mid" else gi.make_water_system(32, 9.0)
    H, S = _device_system(nolsm, system)
    ctx = nolsm.Context()
    _attach_model(nolsm, ctx, system, eval_fp32=True)
    count = 12 if which == "mid" else system.n_mol
    begin = 60 if which == "mid" else 0
    batch = ctx.build_submatrices(H, S, begin, count)
    worst = 0.0
    for local in ([0, count - 1] if which == "mid" else range(0, count, 5)):
        j = begin + local
        nbrs = system.col_idx[system.row_ptr[j]:system.row_ptr[j + 1]]
        for mat, val in ((nolsm.MAT_H, system.h_val), (nolsm.MAT_S, system.s_val)):
            ref = orc.dense_submatrix(system.row_ptr, system.col_idx, val, nbrs)
            got = batch.read(local, mat).cpu().numpy()
            assert np.array_equal(got == 0, ref == 0)
            worst = max(worst, float(np.abs(got - ref).max()))
    assert worst < 1e-6, worst
    ctx.close()


@pytest.mark.parametrize("precision", [1, 0])
def test_density_from_generated_elements(nolsm, mid_system, mid_solution, precision):
    """The whole path (solve at fixed mu) with the model attached reproduces the oracle's D and N_e."""
    system = mid_system
    H, S = _device_system(nolsm, system)
    ctx = nolsm.Context(nolsm.Config(precision=precision))
    _attach_model(nolsm, ctx, system)
    import oracle.nolsm_oracle as orc
    ne, e, D, W, st = ctx.evaluate(H, S, MU, want_w=False)
    sols = mid_solution["solutions"]
    d_ref = orc.density_blocks(sols, system.row_ptr, MU)
    ne_ref = orc.electron_count(sols, MU)
    assert abs(ne - ne_ref) / system.n_mol <= TOL_NE_PER_MOL
    assert np.abs(D.val.cpu().numpy() - d_ref).max() < TOL_D[precision]
    e_ref = orc.electronic_energy_blocks(system.row_ptr, system.col_idx, d_ref, system.h_val)
    assert abs(e - e_ref) / system.n_mol < TOL_E_PER_MOL[precision]
    ctx.close()


def test_model_argument_checks(nolsm, tiny_system):
    import torch
    import nolsm_inputs as gi
    ctx = nolsm.Context()
    pos = torch.as_tensor(tiny_system.pos_q).contiguous().cuda()
    par = gi.model_parameters(tiny_system)
    with pytest.raises(nolsm.NolsmError):
        ctx.set_model(pos, **{**par, "box_q": [par["box_q"][0] + 1] * 3})       # odd box
    with pytest.raises(nolsm.NolsmError):
        ctx.set_model(pos, **{**par, "orb_site": [0, 0, 0, 0, 1, 3]})           # site out of range
    ctx.set_model(pos[:16], **par)                                              # wrong n_mol: caught at build time
    H, S = _device_system(nolsm, tiny_system)
    with pytest.raises(nolsm.NolsmError):
        ctx.build_submatrices(H, S, 0, 4)
    ctx.close()


@pytest.mark.parametrize("precision,tol_x", [(1, 2e-5), (0, 3e-3)])
def test_engine_selection_large_n(nolsm, torch_mod, precision, tol_x):
    """n = 1280 is where the context switches to the pair engine on its own (nolsm.h, NOLSM_FLAG_*): the
    automatic choice and both forced engines must all reproduce sign(A) of the construction, and the automatic
    choice must be bit-identical to the forced pair engine (same kernel, same schedule-independent arithmetic)."""
    import nolsm_inputs as gi
    import oracle.nolsm_oracle as orc
    mats = [gi.make_gapped_symmetric(1280, seed=13, index=i) for i in range(2)]
    a = torch_mod.as_tensor(np.stack([m[0] for m in mats])).cuda()
    scale = torch_mod.as_tensor(np.array([np.abs(m[2]).max() for m in mats], dtype=np.float32)).cuda()
    got = {}
    for flags in (0, nolsm.FLAG_PAIR, nolsm.FLAG_SINGLE):
        ctx = nolsm.Context(nolsm.Config(precision=precision, flags=flags))
        x, stats = ctx.sign_dense_batched(a, scale)
        assert stats.n_unconverged == 0
        for i, (_, q, lam) in enumerate(mats):
            assert np.abs(x[i].cpu().numpy() - orc.sign_by_construction(q, lam)).max() < tol_x
        got[flags] = x.clone()
        ctx.close()
    assert torch_mod.equal(got[0], got[nolsm.FLAG_PAIR])


@pytest.mark.parametrize("precision", [1, 0])
def test_unit_scale_flag_same_result_more_iterations(nolsm, tiny_system, tiny_solution, precision):
    """Readings 5 and 7: the result does not depend on the scale, only the iteration count does.  With
    NOLSM_FLAG_UNIT_SCALE (Y0 = S/bound, X0 = A/bound) D still matches the oracle and no submatrix needs
    fewer iterations than with the centred scaling."""
    import oracle.nolsm_oracle as orc
    sols = tiny_solution["solutions"]
    d_ref = orc.density_blocks(sols, tiny_system.row_ptr, MU)
    H, S = _device_system(nolsm, tiny_system)
    iters = {}
    for flags in (0, nolsm.FLAG_UNIT_SCALE):
        ctx = nolsm.Context(nolsm.Config(precision=precision, flags=flags))
        ne, e, D, W, st = ctx.evaluate(H, S, MU, want_w=False)
        assert np.abs(D.val.cpu().numpy() - d_ref).max() < TOL_D[precision]
        assert abs(ne - orc.electron_count(sols, MU)) / tiny_system.n_mol <= TOL_NE_PER_MOL
        iters[flags] = (st.last.iter_min, st.last.iter_max, st.last.inv_iter_max)
        ctx.close()
    assert iters[nolsm.FLAG_UNIT_SCALE][0] >= iters[0][0] and iters[nolsm.FLAG_UNIT_SCALE][1] >= iters[0][1]
    assert iters[nolsm.FLAG_UNIT_SCALE][2] >= iters[0][2]


@pytest.mark.parametrize("precision", [0, 1])
def test_operator_cache_bitwise_same_as_recomputing(nolsm, mid_system, precision):
    """Several mu steps with the batches streamed through a small workspace: keeping B_j and the own columns
    of S_j^-1 from the first step (nolsm_config.cache_bytes) must give exactly the mu, N and D of redoing
    a1-a3 in every step."""
    import torch
    system = mid_system
    H, S = _device_system(nolsm, system)
    out = {}
    for cache_bytes in (0, -1):
        ctx = nolsm.Context(nolsm.Config(precision=precision, workspace_bytes=384 << 20, cache_bytes=cache_bytes))
        mu, ne, D, st = ctx.solve_mu(H, S, system.n_electrons, -1.2, -0.6, tol_ne_per_mol=-1.0, max_steps=3)
        assert st.resident == 0 and st.n_batches > 1 and st.mu_steps == 3
        assert st.cached == (1 if cache_bytes == 0 else 0)
        out[cache_bytes] = (mu, ne, D.val.clone())
        ctx.close()
    assert out[0][0] == out[-1][0], (out[0][0], out[-1][0])
    assert abs(out[0][1] - out[-1][1]) < 1e-7, (out[0][1], out[-1][1])      # N is summed with FP64 atomics
    assert torch.equal(out[0][2], out[-1][2])


@pytest.mark.parametrize("precision", [0, 1])
def test_gap_hint_scaled_start(nolsm, mid_system, mid_solution, precision):
    """nolsm_config.gap_hint: the scaled Newton-Schulz start gives the oracle's D and N in fewer
    iterations; a hint that is far too large still converges to them."""
    import oracle.nolsm_oracle as orc
    system = mid_system
    sols = mid_solution["solutions"]
    d_ref = orc.density_blocks(sols, system.row_ptr, MU)
    ne_ref = orc.electron_count(sols, MU)
    gap = min(float(np.abs(s.lam - MU).min()) for s in sols)
    H, S = _device_system(nolsm, system)
    iters = {}
    for hint in (0.0, 0.9 * gap, 5.0 * gap):
        ctx = nolsm.Context(nolsm.Config(precision=precision, gap_hint=hint))
        mu, ne, D, st = ctx.solve_mu(H, S, system.n_electrons, 2 * MU, 0.0, tol_ne_per_mol=-1.0, max_steps=1)
        assert st.last.n_unconverged == 0
        assert np.abs(D.val.cpu().numpy() - d_ref).max() < TOL_D[precision]
        assert abs(ne - ne_ref) / system.n_mol <= TOL_NE_PER_MOL
        iters[hint] = st.last.iter_max
        ctx.close()
    assert iters[0.9 * gap] <= iters[0.0] - 2, iters


# ---------------------------------------------------------------------------------------------
# failure surface of the boundary (include/nolsm.h status codes): verdicts come from device counters, with or
# without a stats struct
# ---------------------------------------------------------------------------------------------
def test_status_enoconv_without_stats(nolsm, tiny_system):
    """A sign iteration capped at 2 iterations cannot pass the residual test: NOLSM_ENOCONV from
    nolsm_sign_batched and from nolsm_solve_mu even when no stats struct is passed."""
    H, S = _device_system(nolsm, tiny_system)
    ctx = nolsm.Context(nolsm.Config(max_iter=2))
    batch = ctx.build_submatrices(H, S, 0, 8)
    with pytest.raises(nolsm.NolsmError) as ei:
        ctx.sign_batched(batch, MU, want_stats=False)
    assert ei.value.status == 5
    with pytest.raises(nolsm.NolsmError) as ei:
        ctx.solve_mu(H, S, tiny_system.n_electrons, 2 * MU, 0.0, tol_ne_per_mol=-1.0, max_steps=1, want_stats=False)
    assert ei.value.status == 5
    ctx.close()


def test_status_enotspd(nolsm, tiny_system):
    """An overlap matrix with a negative-definite diagonal block: Eq. 15-17 cannot converge (PAPER.md:203-215
    needs an SPD T_j(S)); the batch that contains the molecule reports NOLSM_ENOTSPD."""
    import torch
    s_bad = tiny_system.s_val.copy()
    k = int(tiny_system.row_ptr[3] + np.searchsorted(tiny_system.col_idx[tiny_system.row_ptr[3]:tiny_system.row_ptr[4]], 3))
    s_bad[k] = -s_bad[k]
    H = nolsm.BlockSparse.from_numpy(tiny_system.row_ptr, tiny_system.col_idx, tiny_system.h_val)
    S = nolsm.BlockSparse(H.row_ptr, H.col_idx, torch.as_tensor(s_bad).contiguous().cuda())
    ctx = nolsm.Context()
    with pytest.raises(nolsm.NolsmError) as ei:
        ctx.solve_mu(H, S, tiny_system.n_electrons, 2 * MU, 0.0, tol_ne_per_mol=-1.0, max_steps=1, want_stats=False)
    assert ei.value.status == 4
    batch = ctx.build_submatrices(H, S, 0, 8)
    with pytest.raises(nolsm.NolsmError) as ei:
        ctx.sign_batched(batch, MU, want_stats=False)
    assert ei.value.status == 4
    ctx.close()


def test_status_ebracket(nolsm, tiny_system):
    """A bracket below the whole spectrum holds no crossing of N(mu) = N_e: NOLSM_EBRACKET."""
    H, S = _device_system(nolsm, tiny_system)
    ctx = nolsm.Context()
    with pytest.raises(nolsm.NolsmError) as ei:
        ctx.solve_mu(H, S, tiny_system.n_electrons, -6.0, -4.0, tol_ne_per_mol=1e-3, max_steps=6)
    assert ei.value.status == 6
    ctx.close()


def test_user_batch_survives_whole_path_calls(nolsm, tiny_system, tiny_solution):
    """A handle from nolsm_build_submatrices stays valid across nolsm_solve_mu / nolsm_sign_dense_batched on the
    same context (those use context-private slots), and a large-then-small sequence of solves does not run out
    of workspace."""
    import torch
    import oracle.nolsm_oracle as orc
    H, S = _device_system(nolsm, tiny_system)
    ctx = nolsm.Context()
    batch = ctx.build_submatrices(H, S, 4, 6)
    ref = batch.read(2, nolsm.MAT_S).clone()
    mu, ne, D, _ = ctx.solve_mu(H, S, tiny_system.n_electrons, -3.0, 0.0, tol_ne_per_mol=1e-3, max_steps=30)
    a = torch.eye(32, dtype=torch.float32).cuda()[None] * 0.5
    ctx.sign_dense_batched(a, None)
    assert torch.equal(batch.read(2, nolsm.MAT_S), ref)
    st = ctx.sign_batched(batch, MU)
    assert st.n_unconverged == 0
    D2 = S.like()
    ne_t = torch.zeros(1, dtype=torch.float64, device="cuda")
    ctx.scatter_density(batch, S, D2, ne_t, None, None)
    d_ref = orc.density_blocks(tiny_solution["solutions"], tiny_system.row_ptr, MU)
    lo, hi = tiny_system.row_ptr[4], tiny_system.row_ptr[10]
    assert np.abs(D2.val.cpu().numpy()[lo:hi] - d_ref[lo:hi]).max() < TOL_D[0]
    ctx.close()


def test_config4_streaming_path_sampled(nolsm):
    """BASELINE configs[3]'s submatrix size and streaming mode at a size the suite can afford: 32,768 molecules at
    the 12 A cutoff (n ~ 1489, the CTA-pair engine, > 100 streamed batches through a 24 GiB workspace), one
    N(mu) evaluation; eight sampled molecules against the oracle and the plateau property for all."""
    import torch
    import nolsm_inputs as gi
    import oracle.nolsm_oracle as orc
    n_mol = 32768
    system = gi.make_water_system(n_mol, 12.0)
    H, S = _device_system(nolsm, system)
    ctx = nolsm.Context(nolsm.Config(precision=0, workspace_bytes=24 << 30))
    q = torch.zeros(n_mol, dtype=torch.float64, device="cuda")
    mu, ne, D, stats = ctx.solve_mu(H, S, system.n_electrons, 2 * MU, 0.0, tol_ne_per_mol=-1.0, max_steps=1, q_mol=q)
    assert stats.n_batches > 100 and stats.last.n_unconverged == 0
    d = D.val.cpu().numpy()
    qh = q.cpu().numpy()
    for j in (0, 300, 5000, 11111, 16384, 23456, 30000, 32767):
        sol = orc.solve_molecule(system.row_ptr, system.col_idx, system.h_val, system.s_val, j)
        assert sol.n > 1400
        ref = sol.density_columns(MU).reshape(-1, 6, 6)
        lo = system.row_ptr[j]
        assert np.abs(d[lo:lo + ref.shape[0]] - ref).max() < TOL_D[0], j
        assert abs(qh[j] - sol.population(MU)) < 5e-3
    assert np.abs(qh - 8.0).max() < 0.03
    assert abs(ne - system.n_electrons) / n_mol < 1e-3
    assert np.isfinite(d).all()
    ctx.close()


# ---------------------------------------------------------------------------------------------
# combined submatrices (section III-B3, Eq. 14)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision", [1, 0])
@pytest.mark.parametrize("which", ["tiny", "w256"])
def test_combined_submatrices_density(nolsm, tiny_system, precision, which):
    """Groups from nolsm_combine_submatrices (bit-exact against the oracle's heuristic), one dense submatrix per
    group through nolsm_build_submatrices_grouped / nolsm_sign_batched / nolsm_scatter_density; every owner's
    blocks D(i, j) and its population against the oracle's solution of the same combined submatrix.
    tiny: the 32-molecule box, where the lists nearly cover the box and the heuristic merges everything into a few
    groups; w256: 256 molecules at 6 A, mostly single molecules plus pairs and triples."""
    import torch
    import nolsm_inputs as gi
    import oracle.nolsm_oracle as orc
    system = tiny_system if which == "tiny" else gi.make_water_system(256, 6.0)
    ref_groups = orc.combine_submatrices(system.row_ptr, system.col_idx)
    own_ptr, own_idx, list_ptr, list_idx = nolsm.combine_submatrices(system.row_ptr, system.col_idx)
    got = [(list(own_idx[own_ptr[g]:own_ptr[g + 1]]), list(list_idx[list_ptr[g]:list_ptr[g + 1]]))
           for g in range(len(own_ptr) - 1)]
    assert got == [(list(o), list(r)) for o, r in ref_groups]
    assert len(got) < system.n_mol
    H, S = _device_system(nolsm, system)
    D = S.like()
    D.val.fill_(float("nan"))
    groups = nolsm.Groups(own_ptr, own_idx, list_ptr, list_idx)
    ctx = nolsm.Context(nolsm.Config(precision=precision))
    batch = ctx.build_submatrices_grouped(H, S, groups, 0, groups.n_groups)
    st = ctx.sign_batched(batch, MU)
    assert st.n_unconverged == 0 and st.n_sub == len(got)
    ne = torch.zeros(1, dtype=torch.float64, device="cuda")
    q = torch.zeros(system.n_mol, dtype=torch.float64, device="cuda")
    ctx.scatter_density(batch, S, D, ne, q, None)
    d = D.val.cpu().numpy()
    assert np.isfinite(d).all()                    # every stored block was written by its owner's group
    qh = q.cpu().numpy()
    checked = 0
    for g, (owners, rows) in enumerate(ref_groups):
        if which == "w256" and len(owners) == 1 and g % 16:
            continue
        sol = orc.solve_group(system.row_ptr, system.col_idx, system.h_val, system.s_val, owners, rows)
        for j in owners:
            ref = sol.density_columns(j, MU).reshape(-1, 6, 6)
            lo = system.row_ptr[j]
            assert np.abs(d[lo:lo + ref.shape[0]] - ref).max() < TOL_D[precision], (g, j)
            checked += 1
    assert checked >= 20
    assert abs(ne.item() - qh.sum()) < 1e-6 * system.n_mol
    assert np.abs(qh - 8.0).max() < 0.05
    ctx.close()


@pytest.mark.parametrize("n,batch", [(200, 3), (512, 2)])
def test_order3_iteration_variant(nolsm, torch_mod, mid_system, mid_solution, n, batch):
    """NOLSM_FLAG_ORDER3 (the third-order Pade member): same sign matrix as the
    construction Q sign(lam) Q^T, fewer iterations than Eq. 9 and the iteration count of the oracle's literal
    restatement; same density matrix as the oracle on a partial batch of the 216-molecule system."""
    import nolsm_inputs as gi
    import oracle.nolsm_oracle as orc
    import torch
    mats = [gi.make_gapped_symmetric(n, seed=23, index=i) for i in range(batch)]
    a = torch_mod.as_tensor(np.stack([m[0] for m in mats])).cuda()
    scale = torch_mod.as_tensor(np.array([np.abs(m[2]).max() for m in mats], dtype=np.float32)).cuda()
    ctx3 = nolsm.Context(nolsm.Config(precision=0, flags=nolsm.FLAG_ORDER3))
    ctx2 = nolsm.Context(nolsm.Config(precision=0))
    x3, st3 = ctx3.sign_dense_batched(a, scale)
    x2, st2 = ctx2.sign_dense_batched(a, scale)
    assert st3.n_unconverged == 0 and st3.iter_max < st2.iter_max
    for i, (am, q, lam) in enumerate(mats):
        assert np.abs(x3[i].cpu().numpy() - orc.sign_by_construction(q, lam)).max() < 3e-3
        _, hist = orc.sign_iteration_order3(am.astype(np.float64), 12, scale=np.abs(lam).max(), history=True)
        k_pass = int(np.argmax(hist < 1e-2))          # first iteration whose residual passes; it is finished ("+1")
        assert st3.iter_min <= k_pass + 1 <= st3.iter_max
    ctx2.close()
    H, S = _device_system(nolsm, mid_system)
    D = S.like()
    batch_h = ctx3.build_submatrices(H, S, 30, 24)
    st = ctx3.sign_batched(batch_h, MU)
    assert st.n_unconverged == 0
    ne_t = torch.zeros(1, dtype=torch.float64, device="cuda")
    ctx3.scatter_density(batch_h, S, D, ne_t, None, None)
    d_ref = orc.density_blocks(mid_solution["solutions"], mid_system.row_ptr, MU)
    lo, hi = mid_system.row_ptr[30], mid_system.row_ptr[54]
    assert np.abs(D.val.cpu().numpy()[lo:hi] - d_ref[lo:hi]).max() < TOL_D[0]
    ctx3.close()


def test_merged_pattern_of_h_and_s(nolsm, mid_system):
    """H0 and S stored on DIFFERENT patterns: S truncated at 6 A, H at 8 A with a seventh of its
    off-diagonal blocks dropped, so neither pattern contains the other.  nolsm_union_pattern + nolsm_expand_store
    give the merged pattern; D on it against the oracle, which slices each matrix from its own store over the
    merged index set."""
    import torch
    import nolsm_inputs as gi
    import oracle.nolsm_oracle as orc
    sys_h = mid_system                                   # 216 molecules, 8 A
    sys_s = gi.make_water_system(216, 6.0)               # same seed -> same positions
    assert np.array_equal(sys_h.pos_q, sys_s.pos_q)
    rows = np.repeat(np.arange(216), np.diff(sys_h.row_ptr))
    keep = (rows == sys_h.col_idx) | ((rows + sys_h.col_idx) % 7 != 0)
    rp_h = np.zeros(217, dtype=np.int32)
    rp_h[1:] = np.cumsum(np.bincount(rows[keep], minlength=216))
    ci_h, h_val = sys_h.col_idx[keep], sys_h.h_val[keep]
    rp_u, ci_u = nolsm.union_pattern(rp_h, ci_h, sys_s.row_ptr, sys_s.col_idx)
    assert len(ci_u) > len(ci_h) and len(ci_u) > sys_s.nnzb
    Hs = nolsm.BlockSparse.from_numpy(rp_h, ci_h, h_val)
    Ss = nolsm.BlockSparse.from_numpy(sys_s.row_ptr, sys_s.col_idx, sys_s.s_val)
    ctx = nolsm.Context(nolsm.Config(precision=1))
    rp_d = torch.as_tensor(rp_u).cuda()
    ci_d = torch.as_tensor(ci_u).cuda()
    H = ctx.expand_store(Hs, rp_d, ci_d)
    S = ctx.expand_store(Ss, rp_d, ci_d)
    begin, count = 40, 16
    batch = ctx.build_submatrices(H, S, begin, count)
    st = ctx.sign_batched(batch, MU)
    assert st.n_unconverged == 0
    D = S.like()
    ne = torch.zeros(1, dtype=torch.float64, device="cuda")
    ctx.scatter_density(batch, S, D, ne, None, None)
    d = D.val.cpu().numpy()
    for j in (begin, begin + 7, begin + count - 1):
        nbrs = ci_u[rp_u[j]:rp_u[j + 1]]
        h_sub = orc.dense_submatrix(rp_h, ci_h, h_val, nbrs)
        s_sub = orc.dense_submatrix(sys_s.row_ptr, sys_s.col_idx, sys_s.s_val, nbrs)
        sol = orc.SubmatrixSolution(j, nbrs, h_sub, s_sub)
        ref = sol.density_columns(MU).reshape(-1, 6, 6)
        assert np.abs(d[rp_u[j]:rp_u[j + 1]] - ref).max() < TOL_D[1]
    ctx.close()
