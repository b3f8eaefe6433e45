"""The C-ABI library builds, loads without a GPU and exports every symbol include/nolsm.h declares.
No compute calls here (there is no GPU on the CPU box); nolsm_create must FAIL loudly without a device."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "nolsm.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    names = set(re.findall(r"\b(nolsm_[a-z0-9_]+)\s*\(", text))
    return sorted(names)


@pytest.fixture(scope="module")
def lib():
    from paper_2104_08245_b200 import build
    build.build()
    import paper_2104_08245_b200 as nolsm
    return nolsm.load_library()


def test_header_declares_the_north_star_entry_points():
    names = _declared_symbols()
    for required in ("nolsm_build_submatrices", "nolsm_sign_batched", "nolsm_scatter_density", "nolsm_solve_mu"):
        assert required in names


def test_library_exports_every_declared_symbol(lib):
    import paper_2104_08245_b200 as nolsm
    declared = _declared_symbols()
    assert declared, "no declarations parsed from include/nolsm.h"
    for name in declared:
        assert hasattr(lib, name), f"libnolsm.so does not export {name}"
    assert sorted(nolsm.EXPORTED_SYMBOLS) == declared


def test_version_and_no_device_behaviour(lib):
    import torch
    assert lib.nolsm_version() >= 1
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    import paper_2104_08245_b200 as nolsm
    with pytest.raises(nolsm.NolsmError) as e:
        nolsm.Context()
    assert e.value.status == 3  # NOLSM_ECUDA: there is no CPU fallback


def test_struct_sizes_match_the_header(lib):
    """ctypes mirrors of the host structs must have the C layout (checked against a tiny C program)."""
    import subprocess
    import tempfile
    import paper_2104_08245_b200.binding as b
    src = r'''
#include <stdio.h>
#include "nolsm.h"
int main(void) { printf("%zu %zu %zu %zu\n", sizeof(nolsm_config), sizeof(nolsm_bsr), sizeof(nolsm_sign_stats),
                        sizeof(nolsm_solve_stats)); return 0; }
'''
    with tempfile.TemporaryDirectory() as d:
        c = os.path.join(d, "s.c")
        open(c, "w").write(src)
        exe = os.path.join(d, "s")
        subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), c, "-o", exe], check=True)
        out = subprocess.run([exe], check=True, capture_output=True, text=True).stdout.split()
    sizes = [int(x) for x in out]
    assert sizes == [ctypes.sizeof(b.Config), ctypes.sizeof(b._Bsr), ctypes.sizeof(b.SignStats),
                     ctypes.sizeof(b.SolveStats)]


def test_combination_heuristic_host_entry_matches_oracle():
    """nolsm_combine_submatrices is host integer work (no device needed): bit-exact groups against the oracle's
    plain-Python restatement of section III-B3 on the hand-built examples of test_oracle_pins.py, on the tiny system
    and on 108- and 256-molecule systems whose lists are far from covering the box (a few pairs and triples merge)."""
    import numpy as np
    import nolsm_inputs as gi
    import oracle.nolsm_oracle as orc
    import paper_2104_08245_b200 as nolsm

    def csr(lists):
        rp = np.zeros(len(lists) + 1, dtype=np.int32)
        rp[1:] = np.cumsum([len(l) for l in lists])
        return rp, np.concatenate([np.asarray(l, dtype=np.int32) for l in lists])

    cases = [csr([[0, 1, 2, 3]] * 4), csr([[0, 1, 2]] * 3 + [[3, 4, 5]] * 3),
             csr([[0, 1], [0, 1, 2], [1, 2, 3], [2, 3, 4], [3, 4]])]
    for n_mol, cutoff in ((32, 6.0), (108, 6.0), (256, 6.0)):
        s = gi.make_water_system(n_mol, cutoff)
        cases.append((s.row_ptr, s.col_idx))
    for rp, ci in cases:
        ref = orc.combine_submatrices(rp, ci)
        own_ptr, own_idx, list_ptr, list_idx = nolsm.combine_submatrices(rp, ci)
        got = [(list(own_idx[own_ptr[g]:own_ptr[g + 1]]), list(list_idx[list_ptr[g]:list_ptr[g + 1]]))
               for g in range(len(own_ptr) - 1)]
        assert got == [(list(o), list(r)) for o, r in ref]
    # the last system has several groups of different sizes (the comparison above is not vacuous)
    assert 1 < len(got) < 256
    # error behaviour: a list that is not ascending
    rp, ci = csr([[1, 0], [0, 1]])
    import pytest
    with pytest.raises(nolsm.NolsmError):
        nolsm.combine_submatrices(rp, ci)


def test_union_pattern_host_entry():
    """nolsm_union_pattern against Python sets (row i kept if H_ij != 0 or S_ij != 0)."""
    import numpy as np
    import paper_2104_08245_b200 as nolsm
    rng = np.random.default_rng(3)
    n = 40
    def rand_pattern(p):
        lists = [sorted(set(np.nonzero(rng.random(n) < p)[0].tolist()) | {i}) for i in range(n)]
        rp = np.zeros(n + 1, dtype=np.int32)
        rp[1:] = np.cumsum([len(l) for l in lists])
        return rp, np.concatenate([np.asarray(l, dtype=np.int32) for l in lists]), lists
    rpa, cia, la = rand_pattern(0.2)
    rpb, cib, lb = rand_pattern(0.1)
    rp, ci = nolsm.union_pattern(rpa, cia, rpb, cib)
    for i in range(n):
        assert list(ci[rp[i]:rp[i + 1]]) == sorted(set(la[i]) | set(lb[i]))
    assert rp[-1] == len(ci)
