"""Property tests (hypothesis) over random tiny inputs: the host-side integer entry points of the C ABI against the
oracle's plain restatements, and invariants of the oracle itself (plan item 4).  CPU only."""
import numpy as np
from hypothesis import given, settings, strategies as st

import oracle.nolsm_oracle as orc
import paper_2104_08245_b200 as nolsm


def _csr(lists):
    rp = np.zeros(len(lists) + 1, dtype=np.int32)
    rp[1:] = np.cumsum([len(l) for l in lists])
    ci = np.concatenate([np.asarray(l, dtype=np.int32) for l in lists]) if lists else np.zeros(0, np.int32)
    return rp, ci


@st.composite
def symmetric_lists(draw, max_n=12):
    """Neighbour lists of a random undirected graph with self loops (what a0 produces: symmetric, self included)."""
    n = draw(st.integers(min_value=1, max_value=max_n))
    bits = draw(st.lists(st.booleans(), min_size=n * (n - 1) // 2, max_size=n * (n - 1) // 2))
    adj = [{i} for i in range(n)]
    k = 0
    for i in range(n):
        for j in range(i + 1, n):
            if bits[k]:
                adj[i].add(j)
                adj[j].add(i)
            k += 1
    return [sorted(a) for a in adj]


@settings(max_examples=150, deadline=None)
@given(symmetric_lists())
def test_combine_submatrices_matches_oracle_on_random_graphs(lists):
    rp, ci = _csr(lists)
    ref = orc.combine_submatrices(rp, ci)
    own_ptr, own_idx, list_ptr, list_idx = nolsm.combine_submatrices(rp, ci)
    got = [(list(own_idx[own_ptr[g]:own_ptr[g + 1]]), list(list_idx[list_ptr[g]:list_ptr[g + 1]]))
           for g in range(len(own_ptr) - 1)]
    assert got == [(list(o), list(r)) for o, r in ref]
    # invariants of section III-B3: a partition of the molecules; every owner's list inside its group's rows;
    # the cubic work never above the one-per-molecule value (every accepted merge satisfies Eq. 14)
    assert sorted(m for o, _ in got for m in o) == list(range(len(lists)))
    for o, r in got:
        for j in o:
            assert set(lists[j]) <= set(r)
    assert sum(len(r) ** 3 for _, r in got) <= sum(len(l) ** 3 for l in lists)


@settings(max_examples=100, deadline=None)
@given(symmetric_lists(max_n=10), symmetric_lists(max_n=10))
def test_union_pattern_is_the_set_union(la, lb):
    n = min(len(la), len(lb))
    la = [[c for c in l if c < n] for l in la[:n]]
    lb = [[c for c in l if c < n] for l in lb[:n]]
    rp, ci = nolsm.union_pattern(*_csr(la), *_csr(lb))
    for i in range(n):
        assert list(ci[rp[i]:rp[i + 1]]) == sorted(set(la[i]) | set(lb[i]))


@settings(max_examples=40, deadline=None)
@given(st.integers(min_value=2, max_value=10), st.integers(min_value=0, max_value=2 ** 31 - 1),
       st.floats(min_value=-0.4, max_value=0.4))
def test_oracle_sign_and_density_identities_on_random_pencils(n, seed, mu):
    """For a random symmetric H and SPD S: sign(S^-1 H - mu)^2 = I, D S D = D, tr(D S) = #(lambda < mu)
    (Eq. 6 / 12), whenever mu is not (numerically) an eigenvalue."""
    rng = np.random.default_rng(seed)
    a = rng.standard_normal((n, n))
    h = 0.5 * (a + a.T)
    b = rng.standard_normal((n, n))
    s = b @ b.T + n * np.eye(n)
    lam, v = orc.generalized_eig(h, s)
    if np.abs(lam - mu).min() < 1e-6:
        return
    sg = orc.sign_from_eig(lam, v, s, mu)
    assert np.abs(sg @ sg - np.eye(n)).max() < 1e-9
    d = orc.density_from_eig(lam, v, mu)
    assert np.abs(d @ s @ d - d).max() < 1e-10
    assert abs(np.trace(d @ s) - (lam < mu).sum()) < 1e-9
    assert np.abs(0.5 * (np.eye(n) - sg) @ np.linalg.inv(s) - d).max() < 1e-9
