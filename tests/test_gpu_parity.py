"""-m gpu parity tests: the CUDA path (through the C ABI) against the oracle, element by element,
on the same seeded inputs.  All integer work: the bar is bit-exact equality."""
import os

import numpy as np
import pytest

import oracle
import workloads

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

GOLD = os.path.join(os.path.dirname(__file__), "golden")


@pytest.fixture(scope="module")
def rna():
    if not torch.cuda.is_available():
        pytest.fail("these tests need a CUDA device (no CPU fallback exists)")
    import paper_1307_7820_b200 as pkg
    return pkg


_ctx_cache = {}


def ctx(pkg, q, engine):
    key = (q, engine)
    if key not in _ctx_cache:
        _ctx_cache[key] = pkg.Rna4r(q, 0, engine)
    return _ctx_cache[key]


def dev_seq(s: bytes):
    return torch.from_numpy(np.frombuffer(s, dtype=np.uint8).copy()).cuda() if len(s) else torch.empty(0, dtype=torch.uint8, device="cuda")


def gpu_table(pkg, r, s: bytes, dtype=None):
    dtype = pkg.TABLE_INT32 if dtype is None else dtype
    score, tab = r.fold(dev_seq(s), len(s), table_dtype=dtype)
    torch.cuda.synchronize()
    return int(score.item()), tab.cpu().numpy()


def rand_seq(rs, n):
    return workloads.ALPHABET.encode()[0:0] + bytes(np.frombuffer(b"ACGU", dtype=np.uint8)[rs.randint(0, 4, size=n)])


# ------------------------------------------------------------------ step a2: the R table
@pytest.mark.parametrize("q", list(range(2, 13)))
def test_rtable_entry_by_entry(rna, q):
    r = rna.Rna4r(q, 0)
    R = r.table()
    want = oracle.rtable(q)
    assert R.shape == want.shape and (R == want).all()
    Rc = r.table_compact()
    assert (Rc == want[::2, ::2]).all()
    r.close()


@pytest.mark.parametrize("q", [9, 10, 11])
def test_ternary_rtable_entry_by_entry(rna, q):
    """Rt[sum_k (v_k - |vbar_k| + 1) 3^(k-1)] == R[v][vbar] for every pair of vectors with bit 0 clear (rna4r.h);
    the pairs reach every one of the 3^(q-1) entries"""
    r = rna.Rna4r(q, 0)
    Rt = r.table_ternary()
    want = oracle.rtable(q)[::2, ::2]
    M = 1 << (q - 1)
    h = np.arange(M, dtype=np.int64)[:, None]
    w = np.arange(M, dtype=np.int64)[None, :]
    idx = np.zeros((M, M), dtype=np.int64)
    for k in range(q - 1):
        idx += (((h >> k) & 1) - ((w >> k) & 1) + 1) * 3 ** k
    assert Rt.shape == (3 ** (q - 1),)
    assert (Rt[idx] == want).all()
    assert np.unique(idx).size == Rt.size
    r.close()
    with pytest.raises(rna.Rna4rError):
        r8 = rna.Rna4r(8, 0)
        try:
            r8.table_ternary()
        finally:
            r8.close()


# ------------------------------------------------------------------ full-table parity, small n
ENGINES = ["tiled", "diag", "paper_tile", "maxplus"]


def engine_id(pkg, name):
    return {"tiled": pkg.ENGINE_TILED, "diag": pkg.ENGINE_DIAG, "paper_tile": pkg.ENGINE_PAPER_TILE,
            "maxplus": pkg.ENGINE_MAXPLUS}[name]


@pytest.mark.parametrize("engine", ENGINES)
@pytest.mark.parametrize("q", list(range(2, 13)))
def test_full_table_all_small_n(rna, engine, q):
    """every n in 0..3q+2 (all residues mod q, n < q, n = 0,1,2) -- SURVEY section 4 tier (iv)"""
    if engine == "tiled" and q > 11:
        pytest.skip("the tiled engine stops at q = 11 (3^11 table bytes do not fit shared memory)")
    r = ctx(rna, q, engine_id(rna, engine))
    rs = np.random.RandomState(1000 + q)
    for n in range(0, 3 * q + 3):
        s = rand_seq(rs, n)
        want_score, want = oracle.nussinov(s, want_table=True)
        if n == 0:
            score, _ = r.fold(dev_seq(s), 0)
            torch.cuda.synchronize()
            assert int(score.item()) == 0
            continue
        got_score, got = gpu_table(rna, r, s)
        assert got_score == want_score, (engine, q, n)
        assert (got == want).all(), (engine, q, n, s)


@pytest.mark.parametrize("engine", ENGINES)
@pytest.mark.parametrize("q", [2, 3, 4, 5, 7, 8, 9, 10, 11])
def test_full_table_tile_boundaries_and_random(rna, engine, q):
    """lengths around the super-tile size T = 8q (ragged tails, several tiles) and random lengths"""
    r = ctx(rna, q, engine_id(rna, engine))
    T = 8 * q
    rs = np.random.RandomState(2000 + q)
    lens = sorted({T - 2, T - 1, T, T + 1, 2 * T - 1, 2 * T, 2 * T + 1, 3 * T + q - 1, 5 * T + 3,
                   int(rs.randint(3 * T, 7 * T)), int(rs.randint(100, 600))})
    for n in lens:
        s = rand_seq(rs, n)
        want_score, want = oracle.nussinov(s, want_table=True)
        for dt in (rna.TABLE_INT32, rna.TABLE_INT16):
            got_score, got = gpu_table(rna, r, s, dt)
            assert got_score == want_score, (engine, q, n)
            assert (got.astype(np.int32) == want).all(), (engine, q, n)


@pytest.mark.parametrize("engine", ENGINES)
def test_structured_sequences(rna, engine):
    """degenerate inputs: one letter, all-pairing hairpins, alternating pairs"""
    r = ctx(rna, 8, engine_id(rna, engine))
    for s in (b"A" * 300, b"A" * 150 + b"U" * 150, b"AU" * 200, b"ACGU" * 90, b"G" * 100 + b"A" * 50 + b"C" * 100,
              b"GGGAAAUCC", b"AGUC"):
        want_score, want = oracle.nussinov(s, want_table=True)
        got_score, got = gpu_table(rna, r, s)
        assert got_score == want_score and (got == want).all(), s[:16]


@pytest.mark.parametrize("engine", ENGINES)
def test_alphabet_and_invalid(rna, engine):
    r = ctx(rna, 4, engine_id(rna, engine))
    for s, want in ((b"acgu" * 10, oracle.nussinov(b"ACGU" * 10)), (b"ACGT" * 10, oracle.nussinov(b"ACGU" * 10))):
        score, _ = r.fold(dev_seq(s))
        torch.cuda.synchronize()
        assert int(score.item()) == want
    score, _ = r.fold(dev_seq(b"ACGUNACGU" * 9))
    torch.cuda.synchronize()
    assert int(score.item()) == -1


# ------------------------------------------------------------------ the five configs
def read_expected(name):
    d = {}
    with open(os.path.join(GOLD, f"{name}_expected.txt")) as f:
        for ln in f:
            if ln.startswith("#"):
                continue
            k, v = ln.split()
            d[k] = v
    cells = np.loadtxt(os.path.join(GOLD, f"{name}_cells.txt"), dtype=np.int64, comments="#")
    return d, cells


def test_cfg1_full_table_q4_int32(rna):
    s = workloads.single_config("cfg1")
    want_score, want = oracle.nussinov(s, want_table=True)
    for eng in (rna.ENGINE_TILED, rna.ENGINE_DIAG, rna.ENGINE_PAPER_TILE, rna.ENGINE_MAXPLUS, rna.ENGINE_SMEM):
        r = ctx(rna, 4, eng)
        got_score, got = gpu_table(rna, r, s, rna.TABLE_INT32)
        assert got_score == want_score == 110
        assert (got == want).all()


def test_cfg2_n2000_q8(rna):
    s = workloads.single_config("cfg2")
    res = oracle.nussinov_fast(s, threads=os.cpu_count() or 1, want_table=True)
    exp, cells = read_expected("cfg2")
    assert res["score"] == int(exp["score"])
    for eng in (rna.ENGINE_TILED, rna.ENGINE_DIAG, rna.ENGINE_PAPER_TILE, rna.ENGINE_MAXPLUS):
        r = ctx(rna, 8, eng)
        got_score, got = gpu_table(rna, r, s, rna.TABLE_INT16)
        assert got_score == res["score"]
        assert (got == res["table"]).all()                       # whole table, not only samples
        assert (got[cells[:, 0] - 1, cells[:, 1] - 1] == cells[:, 2]).all()


def check_large(pkg, name, q, engine):
    s = workloads.single_config(name)
    exp, cells = read_expected(name)
    n = len(s)
    r = ctx(pkg, q, engine)
    # score-only call (the configuration bench.py times) ...
    score, _ = r.fold(dev_seq(s))
    torch.cuda.synchronize()
    assert int(score.item()) == int(exp["score"])
    # ... and the table call: sampled cells from the stored oracle values + properties at any size
    score, tab = r.fold(dev_seq(s), n, table_dtype=pkg.TABLE_INT16)
    torch.cuda.synchronize()
    assert int(score.item()) == int(exp["score"])
    ii = torch.from_numpy(cells[:, 0] - 1).cuda()
    jj = torch.from_numpy(cells[:, 1] - 1).cuda()
    got = tab[ii, jj].cpu().numpy().astype(np.int64)
    assert (got == cells[:, 2]).all()
    assert int(torch.triu(tab).sum(dtype=torch.int64).item()) == int(exp["table_sum"])
    # Lemma 1 on the whole table, on the device
    up = torch.triu(torch.ones((n, n), dtype=torch.bool, device="cuda"), 1)
    dh = (tab[:, 1:] - tab[:, :-1])[up[:, 1:]]
    assert int(dh.min()) >= 0 and int(dh.max()) <= 1
    del dh
    dv = (tab[:-1, :] - tab[1:, :])[up[:-1, :]]
    assert int(dv.min()) >= 0 and int(dv.max()) <= 1
    assert int(torch.tril(tab, -1).abs().max()) == 0 and int(torch.diagonal(tab).abs().max()) == 0


def test_cfg3_n6000_q8(rna):
    check_large(rna, "cfg3", 8, rna.ENGINE_TILED)


def test_cfg3_full_table_elementwise(rna):
    """the whole 6000 x 6000 table, element by element, against the oracle's table (not only samples and sums)"""
    s = workloads.single_config("cfg3")
    res = oracle.nussinov_fast(s, threads=os.cpu_count() or 1, want_table=True)
    r = ctx(rna, 8, rna.ENGINE_TILED)
    score, tab = r.fold(dev_seq(s), len(s), table_dtype=rna.TABLE_INT16)
    torch.cuda.synchronize()
    assert int(score.item()) == res["score"] == 2761
    want = torch.from_numpy(np.ascontiguousarray(res["table"]).astype(np.int16)).cuda()
    assert torch.equal(tab, want), int((tab != want).sum().item())


@pytest.mark.parametrize("engine", ["diag", "paper_tile", "maxplus"])
def test_cfg3_n6000_q8_comparison_engines(rna, engine):
    check_large(rna, "cfg3", 8, engine_id(rna, engine))


@pytest.mark.parametrize("q", [8, 10, 11])
def test_cfg5_n16384(rna, q):
    check_large(rna, "cfg5", q, rna.ENGINE_TILED)


def test_cfg6_n32768_q8(rna):
    """beyond the five configs: n = 32768, score-only call, then the 2 GB int16 table against the
    oracle's stored cells, table sum and Lemma 1"""
    check_large(rna, "cfg6", 8, rna.ENGINE_TILED)


@pytest.mark.parametrize("q", [10, 11])
def test_cfg6_n32768_ternary_q(rna, q):
    """n = 32768 at the q that index the table in base 3 (a 16-bit value field: anchor sums up to n/2 + q fit; the
    binary 18-bit index of q = 10 stopped at n = 32746): the same stored cells, table sum and Lemma 1"""
    check_large(rna, "cfg6", q, rna.ENGINE_TILED)


def test_cfg4_batch_1024(rna):
    seqs, lens = workloads.gc_rich_batch()
    want = np.loadtxt(os.path.join(GOLD, "cfg4_scores.txt"), dtype=np.int64, comments="#")
    assert (want[:, 1] == lens).all()
    flat, offsets, lens32 = workloads.pack_batch(seqs)
    r = ctx(rna, 8, rna.ENGINE_TILED)
    scores = r.fold_batch(torch.from_numpy(flat).cuda(), torch.from_numpy(offsets).cuda(), lens32)
    torch.cuda.synchronize()
    got = scores.cpu().numpy()
    assert (got == want[:, 2]).all()
    assert int(got.sum()) == 231114          # SURVEY 8(c) p9, reproduced by tests/golden/make_golden.py


# ------------------------------------------------------------------ batch and host-buffer edge cases
@pytest.mark.parametrize("engine", ENGINES)
def test_batch_ragged_and_empty(rna, engine):
    r = ctx(rna, 8, engine_id(rna, engine))
    rs = np.random.RandomState(77)
    lens = [0, 1, 2, 7, 8, 9, 63, 64, 65, 0, 127, 128, 129, 200, 333, 1, 0]
    seqs = [rand_seq(rs, n) for n in lens]
    seqs[6] = b"N" + seqs[6][1:]                                   # one invalid sequence
    flat, offsets, lens32 = workloads.pack_batch(seqs)
    scores = r.fold_batch(torch.from_numpy(flat).cuda(), torch.from_numpy(offsets).cuda(), lens32)
    torch.cuda.synchronize()
    got = scores.cpu().numpy()
    want = np.array([oracle.nussinov(s) for s in seqs])
    assert (got == want).all() and got[6] == -1
    # count = 0
    out = r.fold_batch(torch.zeros(1, dtype=torch.uint8, device="cuda"), torch.zeros(1, dtype=torch.int64, device="cuda"),
                       np.zeros(0, dtype=np.int32))
    assert out.numel() == 0


def test_host_variants(rna):
    r = ctx(rna, 8, rna.ENGINE_TILED)
    rs = np.random.RandomState(78)
    s = rand_seq(rs, 300)
    want_score, want = oracle.nussinov(s, want_table=True)
    score, tab = r.fold_host(s, table_dtype=rna.TABLE_INT32)
    assert score == want_score and (tab == want).all()
    seqs = [rand_seq(rs, n) for n in (5, 0, 150, 64, 400)]
    flat, offsets, lens32 = workloads.pack_batch(seqs)
    got = r.fold_batch_host(flat, lens32)
    assert (got == np.array([oracle.nussinov(x) for x in seqs])).all()


def test_error_codes(rna):
    r = ctx(rna, 8, rna.ENGINE_TILED)
    s = dev_seq(b"ACGU" * 50)
    small = torch.empty(256, dtype=torch.uint8, device="cuda")
    with pytest.raises(rna.Rna4rError) as e:
        r.fold(s, workspace=small)
    assert e.value.code == -4
    with pytest.raises(rna.Rna4rError) as e:
        r.fold(s, n=-1)
    assert e.value.code == -3
    r12 = rna.Rna4r(12, 0)
    assert r12.engine == rna.ENGINE_DIAG
    with pytest.raises(rna.Rna4rError) as e:
        r12.set_engine(rna.ENGINE_TILED)
    assert e.value.code == -9
    sc, _ = r12.fold(dev_seq(workloads.uniform_sequence(5, 150)))
    torch.cuda.synchronize()
    assert int(sc.item()) == oracle.nussinov(workloads.uniform_sequence(5, 150))
    r12.close()


def test_determinism_repeat_calls(rna):
    r = ctx(rna, 8, rna.ENGINE_TILED)
    s = dev_seq(workloads.uniform_sequence(9, 1500))
    a, ta = r.fold(s, table_dtype=rna.TABLE_INT16)
    ta = ta.clone()
    for _ in range(3):
        b, tb = r.fold(s, table_dtype=rna.TABLE_INT16)
        torch.cuda.synchronize()
        assert int(a.item()) == int(b.item()) and torch.equal(ta, tb)


# ------------------------------------------------------------------ pipelined closures, late products, q sweep
@pytest.mark.parametrize("q", [5, 8, 9, 10, 11])
def test_midsize_scores_every_late_product_shape(rna, q):
    """lengths of 2..9 super-tiles per side: super-tile diagonals dp = 1 (no late product), 2 (one block, both
    operands arriving), 3 (two late blocks, no bulk stage) and >= 4 (bulk stages + late blocks); sampled cells
    against the fast oracle"""
    r = ctx(rna, q, rna.ENGINE_TILED)
    T = 8 * q
    rs = np.random.RandomState(4000 + q)
    for nt in (2, 3, 4, 5, 7, 9):
        n = nt * T - int(rs.randint(0, T))
        s = rand_seq(rs, n)
        cells = np.stack([rs.randint(1, n + 1, size=400), rs.randint(1, n + 1, size=400)], axis=1).astype(np.int32)
        cells.sort(axis=1)
        want = oracle.nussinov_fast(s, threads=4, cells=cells)
        score, tab = r.fold(dev_seq(s), table_dtype=rna.TABLE_INT16)
        torch.cuda.synchronize()
        assert int(score.item()) == want["score"], (q, n)
        got = tab.cpu().numpy()[cells[:, 0] - 1, cells[:, 1] - 1]
        assert (got == want["cells"]).all(), (q, n)


def test_skewed_base_distributions(rna):
    """long runs of equal difference vectors (all-zero, all-one) and rare pairs: sequences far from uniform"""
    r = ctx(rna, 8, rna.ENGINE_TILED)
    rs = np.random.RandomState(77)
    for p in ([0.97, 0.01, 0.01, 0.01], [0.49, 0.01, 0.01, 0.49], [0.05, 0.45, 0.45, 0.05], [0.7, 0.0, 0.0, 0.3]):
        n = int(rs.randint(500, 900))
        s = bytes(rs.choice(list(b"ACGU"), size=n, p=p).tolist())
        want_score, want = oracle.nussinov(s, want_table=True)
        got_score, got = gpu_table(rna, r, s, rna.TABLE_INT16)
        assert got_score == want_score and (got.astype(np.int32) == want).all(), p


@pytest.mark.parametrize("q", [4, 9, 10, 11])
def test_batch_other_q(rna, q):
    r = ctx(rna, q, rna.ENGINE_TILED)
    seqs, _ = workloads.random_sequences(500 + q, 40, 0, 450)
    flat, offsets, lens = workloads.pack_batch(seqs)
    got = r.fold_batch(torch.from_numpy(flat).cuda(), torch.from_numpy(offsets).cuda(), lens)
    torch.cuda.synchronize()
    assert (got.cpu().numpy() == np.array([oracle.nussinov(x) for x in seqs])).all()


def test_length_limit_of_the_word_format(rna):
    """every q keeps a 16-bit value field below the index field (q >= 9: base-3 index): the ABI's n <= 65534 holds"""
    r10 = ctx(rna, 10, rna.ENGINE_TILED)
    lim = 65534
    assert r10.workspace_bytes(lim) > 0
    with pytest.raises(rna.Rna4rError) as e:
        r10.fold(dev_seq(b"A" * 16), n=lim + 1, workspace=torch.empty(1 << 20, dtype=torch.uint8, device="cuda"))
    assert e.value.code == -3
