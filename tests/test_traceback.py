"""Traceback.  Several optimal structures may exist, so the CUDA result is
compared on what is unique -- the number of pairs, D(1,n) -- and checked for feasibility against the
definition (oracle/structure.py check_structure); the oracle's own traceback is pinned the same way."""
import numpy as np
import pytest

import oracle
import workloads
from oracle import structure


# ------------------------------------------------------------------ CPU: the checker and the oracle traceback
def test_checker_accepts_and_rejects_by_the_definition():
    assert structure.check_structure("GGGAAACCC", [8, 7, 6, -1, -1, -1, 2, 1, 0]) == 3      # hairpin
    assert structure.check_structure("ACGU", [-1, -1, -1, -1]) == 0
    assert structure.check_structure("ACGT", [3, 2, 1, 0]) == 2                                  # T == U, nested
    with pytest.raises(AssertionError):
        structure.check_structure("AUAU", [2, 3, 0, 1])            # (0,2) is A-A: not complementary
    with pytest.raises(AssertionError):
        structure.check_structure("ACUG", [2, 3, 0, 1])            # (0,2),(1,3) complementary but crossing
    with pytest.raises(AssertionError):
        structure.check_structure("AUU", [1, 0, 0])                # base 0 in two pairs / not symmetric
    with pytest.raises(AssertionError):
        structure.check_structure("GU", [1, 0])                    # wobble pair: not in the paper's pair set (g1)


def test_oracle_traceback_is_feasible_and_optimal_small():
    rs = np.random.RandomState(5)
    for n in list(range(0, 14)) + [20, 33, 64, 100]:
        for _ in range(4):
            s = bytes(rs.choice(list(b"ACGU"), size=n).tolist())
            score, tab = oracle.nussinov(s, want_table=True)
            part = structure.traceback(s, tab)
            assert structure.check_structure(s, part) == score
            if n <= 12:
                assert score == oracle.brute_force_matchings(s)    # the count is the brute-force optimum


# ------------------------------------------------------------------ GPU
gpu = pytest.mark.gpu


@pytest.fixture(scope="module")
def rna():
    import torch
    import paper_1307_7820_b200 as pkg
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    return pkg


def _fold_and_trace(pkg, r, seq: bytes, dt):
    import torch
    n = len(seq)
    d = torch.from_numpy(np.frombuffer(seq, dtype=np.uint8).copy()).cuda() if n else torch.empty(0, dtype=torch.uint8, device="cuda")
    score, tab = r.fold(d, n, table_dtype=dt) if n else (None, torch.empty((0, 0), dtype=torch.int16, device="cuda"))
    pairs, npairs = r.traceback(d, tab, n)
    torch.cuda.synchronize()
    return (int(score.item()) if n else 0), pairs.cpu().numpy(), int(npairs.item())


@gpu
@pytest.mark.parametrize("q", [4, 8, 10])
def test_traceback_small_and_tile_boundaries(rna, q):
    r = rna.Rna4r(q, 0)
    rs = np.random.RandomState(300 + q)
    T = 8 * q
    for n in [0, 1, 2, 3, 7, T - 1, T, T + 1, 3 * T + 5, int(rs.randint(200, 700))]:
        s = bytes(rs.choice(list(b"ACGU"), size=n).tolist())
        want = oracle.nussinov(s)
        for dt in (rna.TABLE_INT16, rna.TABLE_INT32):
            score, pairs, npairs = _fold_and_trace(rna, r, s, dt)
            assert score == want and npairs == want, (q, n)
            assert structure.check_structure(s, pairs) == want, (q, n)


@gpu
def test_traceback_structured_and_deterministic(rna):
    r = rna.Rna4r(8, 0)
    for s in (b"A" * 200, b"A" * 150 + b"U" * 150, b"AU" * 200, b"G" * 100 + b"A" * 50 + b"C" * 100, b"GGGAAAUCC"):
        want = oracle.nussinov(s)
        score, pairs, npairs = _fold_and_trace(rna, r, s, rna.TABLE_INT16)
        assert npairs == want and structure.check_structure(s, pairs) == want
        _, pairs2, _ = _fold_and_trace(rna, r, s, rna.TABLE_INT16)
        assert (pairs == pairs2).all()                       # the rule (pair first, smallest k) is deterministic


@gpu
def test_traceback_matches_the_oracle_rule_on_small_inputs(rna):
    """The oracle traceback applies the same rule (pair first, then the smallest k), so on the same table the
    two structures are identical, not merely equivalent."""
    r = rna.Rna4r(8, 0)
    rs = np.random.RandomState(77)
    for n in (30, 65, 130, 257):
        s = bytes(rs.choice(list(b"ACGU"), size=n).tolist())
        _, tab = oracle.nussinov(s, want_table=True)
        _, pairs, _ = _fold_and_trace(rna, r, s, rna.TABLE_INT32)
        assert (pairs == structure.traceback(s, tab)).all(), n


@gpu
def test_traceback_invalid_sequence_and_errors(rna):
    import torch
    r = rna.Rna4r(8, 0)
    s = b"ACGUNACGU" * 9
    d = torch.from_numpy(np.frombuffer(s, dtype=np.uint8).copy()).cuda()
    _, tab = r.fold(d, table_dtype=rna.TABLE_INT16)
    _, npairs = r.traceback(d, tab)
    torch.cuda.synchronize()
    assert int(npairs.item()) == -1
    L = r.lib
    one = torch.zeros(16, dtype=torch.int32, device="cuda")
    assert L.rna4r_traceback(r.h, d.data_ptr(), len(s), tab.data_ptr(), rna.TABLE_INT16, one.data_ptr(), one.data_ptr(), one.data_ptr(), 8, None) == -4
    assert L.rna4r_traceback(r.h, d.data_ptr(), len(s), tab.data_ptr(), 0, one.data_ptr(), one.data_ptr(), one.data_ptr(), 1 << 20, None) == -8
    assert L.rna4r_traceback(r.h, None, len(s), tab.data_ptr(), rna.TABLE_INT16, one.data_ptr(), one.data_ptr(), one.data_ptr(), 1 << 20, None) == -2


@gpu
def test_traceback_cfg2_and_cfg3(rna):
    """full sizes: feasibility by the O(n) checker, count against the stored expected D(1,n)"""
    r = rna.Rna4r(8, 0)
    for name, want in (("cfg2", 917), ("cfg3", 2761)):
        s = workloads.single_config(name)
        score, pairs, npairs = _fold_and_trace(rna, r, s, rna.TABLE_INT16)
        assert score == want and npairs == want
        assert structure.check_structure(s, pairs) == want
