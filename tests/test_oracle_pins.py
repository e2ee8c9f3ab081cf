"""Pins for the oracle (oracle/) against what the paper and the mathematics fix -- no CUDA here.

p1 brute force (definition), p2/p3 hand-worked values (tests/golden/), p4 closed
forms, p5 invariants (Lemma 1), p6 symmetries, four-term == two-term form,
fast-plain == plain, Algorithm 1 == plain, p7 R-table pins.
"""
import itertools
import os

import numpy as np
import pytest

import oracle
import workloads

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def rand_seq(rs, n, alphabet="ACGU"):
    return "".join(alphabet[c] for c in rs.randint(0, len(alphabet), size=n))


# ---------------------------------------------------------------- p1: brute force
def test_p1_all_strings_up_to_7_match_both_enumerators():
    for n in range(0, 8):
        for tup in itertools.product("ACGU", repeat=n):
            s = "".join(tup)
            d = oracle.nussinov(s)
            assert d == oracle.brute_force_matchings(s), s
            assert d == oracle.brute_force_structural(s), s


def test_p1_random_strings_to_12():
    rs = np.random.RandomState(101)
    for n in range(8, 13):
        for _ in range(40):
            s = rand_seq(rs, n)
            d = oracle.nussinov(s)
            assert d == oracle.brute_force_matchings(s) == oracle.brute_force_structural(s), s


def test_p1_every_cell_is_brute_force_of_its_substring():
    rs = np.random.RandomState(102)
    for n in (5, 7, 9):
        for _ in range(12):
            s = rand_seq(rs, n)
            _, tab = oracle.nussinov(s, want_table=True)
            for i in range(1, n + 1):
                for j in range(i, n + 1):
                    assert tab[i - 1, j - 1] == oracle.brute_force_matchings(s[i - 1:j]), (s, i, j)
            assert (np.tril(tab, -1) == 0).all()


# ---------------------------------------------------------------- p2 / p3: hand-worked fixtures
def test_p2_hand_worked_scores():
    with open(os.path.join(GOLD, "worked_examples.txt")) as f:
        rows = [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]
    assert len(rows) >= 16
    for r in rows:
        s = "" if r[0] == "-" else r[0]
        assert oracle.nussinov(s) == int(r[1]), s
        assert oracle.brute_force_matchings(s) == int(r[1]), s


def test_p3_hand_worked_tables():
    with open(os.path.join(GOLD, "worked_tables.txt")) as f:
        lines = [ln.strip() for ln in f if ln.strip() and not ln.startswith("#")]
    k = 0
    seen = 0
    while k < len(lines):
        s = lines[k]
        n = len(s)
        _, tab = oracle.nussinov(s, want_table=True)
        for i in range(1, n + 1):
            want = [int(x) for x in lines[k + i].split()]
            assert list(tab[i - 1, i - 1:]) == want, (s, i)
        k += n + 1
        seen += 1
    assert seen == 2


# ---------------------------------------------------------------- p4: closed forms
def test_p4_closed_forms():
    for a in range(0, 7):
        for b in range(0, 7):
            s = "A" * a + "U" * b
            _, tab = oracle.nussinov(s, want_table=True)
            for i in range(1, a + b + 1):
                for j in range(i, a + b + 1):
                    sub = s[i - 1:j]
                    assert tab[i - 1, j - 1] == min(sub.count("A"), sub.count("U"))
    for m in range(0, 9):
        assert oracle.nussinov("AU" * m) == m
        assert oracle.nussinov("ACGU" * m) == 2 * m
    rs = np.random.RandomState(7)
    for alpha in ("AC", "AG", "UC", "UG", "A", "G"):
        s = rand_seq(rs, 60, alpha)
        _, tab = oracle.nussinov(s, want_table=True)
        assert (tab == 0).all()


# ---------------------------------------------------------------- p5: invariants
def check_invariants(s, tab):
    n = len(s)
    t = tab.astype(np.int64)
    assert (np.diag(t) == 0).all()                                   # D(i,i) = 0
    assert (np.tril(t, -1) == 0).all()
    up = np.triu(np.ones((n, n), dtype=bool), 1)
    dh = t[:, 1:] - t[:, :-1]                                        # D(i,j) - D(i,j-1)
    assert set(np.unique(dh[up[:, 1:]])) <= {0, 1}
    dv = t[:-1, :] - t[1:, :]                                        # D(i,j) - D(i+1,j)
    assert set(np.unique(dv[up[:-1, :]])) <= {0, 1}
    # upper bounds: floor(len/2) and min(#A,#U)+min(#C,#G)
    cnt = {c: np.concatenate([[0], np.cumsum([ch == c for ch in s])]) for c in "ACGU"}
    for i in range(1, n + 1, max(1, n // 25)):
        for j in range(i, n + 1, max(1, n // 25)):
            c = {k: cnt[k][j] - cnt[k][i - 1] for k in "ACGU"}
            assert t[i - 1, j - 1] <= (j - i + 1) // 2
            assert t[i - 1, j - 1] <= min(c["A"], c["U"]) + min(c["C"], c["G"])
    # superadditivity D(i,j) >= D(i,k) + D(k+1,j) on sampled triples
    rs = np.random.RandomState(n)
    for _ in range(300):
        i, k, j = sorted(rs.randint(1, n + 1, size=3))
        if k < j:
            assert t[i - 1, j - 1] >= t[i - 1, k - 1] + t[k, j - 1]


def test_p5_invariants_lemma1():
    rs = np.random.RandomState(5)
    for n in (1, 2, 3, 17, 64, 150):
        s = rand_seq(rs, n)
        _, tab = oracle.nussinov(s, want_table=True)
        check_invariants(s, tab)


# ---------------------------------------------------------------- p6: symmetries
def test_p6_reversal_and_complement():
    rs = np.random.RandomState(6)
    comp = str.maketrans("ACGU", "UGCA")
    for n in (9, 33, 80):
        s = rand_seq(rs, n)
        _, tab = oracle.nussinov(s, want_table=True)
        _, trev = oracle.nussinov(s[::-1], want_table=True)
        _, tcmp = oracle.nussinov(s.translate(comp), want_table=True)
        assert (tcmp == tab).all()
        # D_rev(n+1-j, n+1-i) = D(i,j)  <=> trev flipped on both axes and transposed
        assert (trev[::-1, ::-1].T == tab).all()


def test_case_and_T_and_invalid():
    assert oracle.nussinov("acgu") == oracle.nussinov("ACGU") == 2
    assert oracle.nussinov("ACGT") == 2
    assert oracle.nussinov("ACGN") == -1
    assert oracle.nussinov("AC U") == -1


# ---------------------------------------------------------------- forms and storage modes agree
def test_fourterm_form_equals_eq1():
    rs = np.random.RandomState(8)
    for n in (0, 1, 2, 5, 31, 120):
        s = rand_seq(rs, n)
        a, ta = oracle.nussinov(s, want_table=True)
        b, tb = oracle.nussinov_fourterm(s, want_table=True)
        assert a == b and (ta == tb).all()


def test_fast_plain_equals_plain():
    rs = np.random.RandomState(9)
    for n, th in ((0, 1), (1, 1), (2, 2), (77, 1), (300, 3), (801, 4)):
        s = rand_seq(rs, n)
        a, ta = oracle.nussinov(s, want_table=True)
        cells = workloads.sample_cells(n, 8, 50) if n >= 10 else None
        r = oracle.nussinov_fast(s, threads=th, cells=cells, want_table=True, want_sum=True)
        assert r["score"] == a
        assert (r["table"] == ta).all()
        assert r["table_sum"] == int(np.triu(ta).sum())
        if cells is not None:
            assert (r["cells"] == ta[cells[:, 0] - 1, cells[:, 1] - 1]).all()


def test_config1_and_2_values_and_generator():
    s1 = workloads.single_config("cfg1")
    assert s1[:24] == b"AUCAUUUUCUCGAUGAAAGCGUUG"
    sc, tab = oracle.nussinov(s1, want_table=True)
    check_invariants(s1.decode(), tab)
    # SURVEY.md 8(c) p9 provisional values from an independent throwaway implementation
    assert sc == 110 and int(tab.sum()) == 1169524 and tab[0, 127] == 54 and tab[128, 255] == 54


# ---------------------------------------------------------------- p8: Algorithm 1 == plain
@pytest.mark.parametrize("q", list(range(2, 11)))
def test_p8_algorithm1_equals_plain_all_small_n(q):
    rs = np.random.RandomState(80 + q)
    for n in range(0, 3 * q + 3):
        s = rand_seq(rs, n)
        a, ta = oracle.nussinov(s, want_table=True)
        r = oracle.two_vector_serial(s, q, want_table=True)
        assert r["score"] == a, (q, n, s)
        assert (r["table"] == ta).all(), (q, n, s)


def test_p8_algorithm1_equals_plain_random_to_600():
    rs = np.random.RandomState(81)
    for q, n in ((2, 97), (3, 200), (4, 256), (5, 333), (8, 600), (9, 410), (10, 555), (12, 300)):
        s = rand_seq(rs, n)
        a, ta = oracle.nussinov(s, want_table=True)
        r = oracle.two_vector_serial(s, q, want_table=True)
        assert r["score"] == a and (r["table"] == ta).all()
        assert r["lookups"] > 0


# ---------------------------------------------------------------- p8': the other serial variants
@pytest.mark.parametrize("variant", ["partially_memoized", "completely_memoized", "frid_gusfield"])
@pytest.mark.parametrize("q", [2, 3, 4, 5, 8])
def test_p8_serial_variants_equal_plain_all_small_n(variant, q):
    rs = np.random.RandomState(85 + q)
    for n in range(0, 3 * q + 3):
        s = rand_seq(rs, n)
        a, ta = oracle.nussinov(s, want_table=True)
        r = oracle.serial_variant(s, q, variant, want_table=True)
        assert r["score"] == a, (variant, q, n, s)
        assert (r["table"] == ta).all(), (variant, q, n, s)


def test_p8_serial_variants_random_and_preprocessing_work():
    """whole tables against eq. (1); the memoised variants preprocess no more than the exhaustive 2^2q pairs
    (PAPER.md:219), the completely memoised one no more than the partially memoised one, and FG does
    2^q evaluations for every group of every row ("duplicated work")"""
    rs = np.random.RandomState(86)
    for q, n in ((3, 211), (4, 256), (5, 333), (8, 500)):
        s = rand_seq(rs, n)
        a, ta = oracle.nussinov(s, want_table=True)
        res = {v: oracle.serial_variant(s, q, v, want_table=True) for v in oracle.SERIAL_VARIANTS}
        tv = oracle.two_vector_serial(s, q)
        for v, r in res.items():
            assert r["score"] == a and (r["table"] == ta).all(), (v, q, n)
            assert r["lookups"] == tv["lookups"]
        pm, cm, fg = res["partially_memoized"], res["completely_memoized"], res["frid_gusfield"]
        assert 0 < cm["blackbox_evals"] <= pm["blackbox_evals"] <= 4 ** q
        assert pm["blackbox_evals"] % (1 << q) == 0
        assert fg["blackbox_evals"] > pm["blackbox_evals"] and fg["blackbox_evals"] % (1 << q) == 0
    assert oracle.serial_variant(b"ACGN", 4, "frid_gusfield")["score"] == -1


# ---------------------------------------------------------------- p7: R table
@pytest.mark.parametrize("q", [2, 3, 4, 5, 8, 10])
def test_p7_rtable_pins(q):
    R = oracle.rtable(q).astype(np.int64)
    N = 1 << q
    pop = np.array([bin(v).count("1") for v in range(N)])
    assert R.min() >= 0 and R.max() <= q
    assert (R[:, 0] == pop).all()                 # vbar = 0: the max is the last running total
    assert (R[0, :] == 0).all()                   # v = 0: never above the initial max-val 0
    assert (np.diag(R) == 0).all()                # same bit pattern: V_p + Vbar_p == 0 for all p
    for k in range(q):                            # monotone: a v bit never lowers, a vbar bit never raises
        bit = 1 << k
        idx = np.array([v for v in range(N) if not v & bit])
        assert (R[idx | bit, :] >= R[idx, :]).all()
        assert (R[:, idx | bit] <= R[:, idx]).all()
    # direct use of eq. (3): for random monotone runs, D(i,l)+D(l+1,j)+R[v][vbar] == max_k D(i,k-1)+D(k,j)
    rs = np.random.RandomState(q)
    for _ in range(200):
        hv = rs.randint(0, 2, size=q); hv[0] = 0
        vv = rs.randint(0, 2, size=q); vv[0] = 0
        row = 5 + np.cumsum(hv)                   # D(i,l+p),  p = 0..q-1
        col = 9 - np.cumsum(vv)                   # D(l+1+p,j), p = 0..q-1
        v = int(sum(int(b) << p for p, b in enumerate(hv)))
        w = int(sum(int(b) << p for p, b in enumerate(vv)))
        assert row[0] + col[0] + R[v, w] == int((row + col).max())
        val, idx = oracle.blackbox(q, v, w)
        assert val == R[v, w] and (row + col)[idx] == (row + col).max()
        assert idx == int(np.argmax(row + col))   # strict '>' keeps the smallest index (reading g11)
