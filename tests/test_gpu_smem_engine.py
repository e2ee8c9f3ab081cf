"""-m gpu parity tests of RNA4R_ENGINE_SMEM (one CTA per sequence, state in shared memory):
full tables against the plain oracle for every small n and every supported q, lengths around the strip / tile
boundaries up to the engine's limit, the batch of config 4 through the AUTO routing, ragged / empty / invalid
batches, and the fallback to the tiled engine when a sequence does not fit."""
import os

import numpy as np
import pytest

import oracle
import workloads

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

GOLD = os.path.join(os.path.dirname(__file__), "golden")
QS = [4, 5, 6, 7, 8]


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


def rand_seq(rs, n):
    return bytes(np.frombuffer(b"ACGU", dtype=np.uint8)[rs.randint(0, 4, size=n)])


def gpu_table(pkg, r, s: bytes, dtype=None):
    dtype = pkg.TABLE_INT32 if dtype is None else dtype
    score, tab = r.fold(dev_seq(s), len(s), table_dtype=dtype)
    torch.cuda.synchronize()
    return int(score.item()), tab.cpu().numpy()


@pytest.mark.parametrize("q", QS)
def test_full_table_all_small_n(rna, q):
    """every n in 0..6q+2: all residues mod q, n < q, one to six tiles per side, strips of 4 tiles with ragged ends"""
    r = ctx(rna, q, rna.ENGINE_SMEM)
    rs = np.random.RandomState(7000 + q)
    for n in range(0, 6 * q + 3):
        s = rand_seq(rs, n)
        want_score, want = oracle.nussinov(s, want_table=True)
        if n == 0:
            score, _ = r.fold(dev_seq(s), 0)
            torch.cuda.synchronize()
            assert int(score.item()) == 0
            continue
        got_score, got = gpu_table(rna, r, s)
        assert got_score == want_score, (q, n)
        assert (got == want).all(), (q, n, s)


@pytest.mark.parametrize("q", QS)
def test_full_table_strip_boundaries_and_random(rna, q):
    """lengths around multiples of the strip width 4q (first bulk, first early bulk, split early bulk) and random
    lengths up to the engine's limit, both table types"""
    r = ctx(rna, q, rna.ENGINE_SMEM)
    lim = r.smem_max_n()
    assert lim >= 300
    S = 4 * q
    rs = np.random.RandomState(7100 + q)
    lens = sorted({S - 1, S, S + 1, 2 * S - 1, 2 * S + 1, 3 * S, 5 * S + 3, 9 * S - 1, 12 * S + q - 1,
                   int(rs.randint(3 * S, 14 * S)), int(rs.randint(100, 600)), min(lim, 640), lim})
    for n in lens:
        if n > lim:
            continue
        s = rand_seq(rs, n)
        res = oracle.nussinov_fast(s, threads=os.cpu_count() or 1, want_table=True)
        for dt in ((rna.TABLE_INT32, rna.TABLE_INT16) if n < 300 else (rna.TABLE_INT16,)):
            got_score, got = gpu_table(rna, r, s, dt)
            assert got_score == res["score"], (q, n)
            assert (got.astype(np.int32) == res["table"]).all(), (q, n)


def test_structured_and_skewed_sequences(rna):
    r = ctx(rna, 8, rna.ENGINE_SMEM)
    rs = np.random.RandomState(7200)
    cases = [b"A" * 300, b"A" * 150 + b"U" * 150, b"AU" * 200, b"ACGU" * 90, b"G" * 100 + b"A" * 50 + b"C" * 100,
             b"GGGAAAUCC", b"AGUC"]
    for p in ([0.97, 0.01, 0.01, 0.01], [0.49, 0.01, 0.01, 0.49], [0.05, 0.45, 0.45, 0.05], [0.7, 0.0, 0.0, 0.3]):
        cases.append(bytes(rs.choice(list(b"ACGU"), size=int(rs.randint(400, 700)), p=p).tolist()))
    for s in cases:
        want_score, want = oracle.nussinov(s, want_table=True)
        got_score, got = gpu_table(rna, r, s)
        assert got_score == want_score and (got == want).all(), s[:16]


def test_alphabet_and_invalid(rna):
    r = ctx(rna, 4, rna.ENGINE_SMEM)
    for s, want in ((b"acgu" * 10, oracle.nussinov(b"ACGU" * 10)), (b"ACGT" * 10, oracle.nussinov(b"ACGU" * 10))):
        score, _ = r.fold(dev_seq(s))
        torch.cuda.synchronize()
        assert int(score.item()) == want
    score, _ = r.fold(dev_seq(b"ACGUNACGU" * 9))
    torch.cuda.synchronize()
    assert int(score.item()) == -1


@pytest.mark.parametrize("engine", ["auto", "smem"])
def test_cfg4_batch_1024(rna, engine):
    """config 4 through the routing a user gets (AUTO -> SMEM engine: one launch) and with the engine forced"""
    seqs, lens = workloads.gc_rich_batch()
    want = np.loadtxt(os.path.join(GOLD, "cfg4_scores.txt"), dtype=np.int64, comments="#")
    assert (want[:, 1] == lens).all()
    flat, offsets, lens32 = workloads.pack_batch(seqs)
    r = ctx(rna, 8, rna.ENGINE_AUTO if engine == "auto" else rna.ENGINE_SMEM)
    assert int(lens32.max()) <= r.smem_max_n()
    scores = r.fold_batch(torch.from_numpy(flat).cuda(), torch.from_numpy(offsets).cuda(), lens32)
    torch.cuda.synchronize()
    assert r.last_launch_count() == 1                     # the SMEM engine: a single kernel for the whole batch
    got = scores.cpu().numpy()
    assert (got == want[:, 2]).all()
    assert int(got.sum()) == 231114


@pytest.mark.parametrize("q", QS)
def test_batch_ragged_empty_invalid(rna, q):
    r = ctx(rna, q, rna.ENGINE_SMEM)
    rs = np.random.RandomState(7300 + q)
    lens = [0, 1, 2, q - 1, q, q + 1, 4 * q - 1, 4 * q, 4 * q + 1, 0, 127, 128, 129, 200, 333, 1, 0, 450]
    seqs = [rand_seq(rs, n) for n in lens]
    seqs[6] = b"N" + seqs[6][1:]                                   # one invalid sequence
    flat, offsets, lens32 = workloads.pack_batch(seqs)
    status = torch.full((len(seqs),), -7, dtype=torch.int32, device="cuda")
    scores = r.fold_batch(torch.from_numpy(flat).cuda(), torch.from_numpy(offsets).cuda(), lens32, status_out=status)
    torch.cuda.synchronize()
    got = scores.cpu().numpy()
    want = np.array([oracle.nussinov(s) for s in seqs])
    assert (got == want).all() and got[6] == -1
    st = status.cpu().numpy()
    assert st[6] == 1 and (np.delete(st, 6) == 0).all()
    out = r.fold_batch(torch.zeros(1, dtype=torch.uint8, device="cuda"), torch.zeros(1, dtype=torch.int64, device="cuda"),
                       np.zeros(0, dtype=np.int32))
    assert out.numel() == 0


def test_bad_offsets_status(rna):
    r = ctx(rna, 8, rna.ENGINE_SMEM)
    rs = np.random.RandomState(7400)
    seqs = [rand_seq(rs, n) for n in (50, 60, 70)]
    flat, offsets, lens32 = workloads.pack_batch(seqs)
    offsets = offsets.copy()
    offsets[2] -= 3                                                # sequences 1 and 2 disagree with lens_host
    status = torch.zeros(3, dtype=torch.int32, device="cuda")
    scores = r.fold_batch(torch.from_numpy(flat).cuda(), torch.from_numpy(offsets).cuda(), lens32, status_out=status)
    torch.cuda.synchronize()
    assert scores.cpu().numpy().tolist() == [oracle.nussinov(seqs[0]), -1, -1]
    assert status.cpu().numpy().tolist() == [0, 2, 2]


def test_auto_splits_a_batch_between_the_engines(rna):
    """sequences beyond the shared-memory limit run on the tiled engine (5 launches), the rest of the same batch on the
    SMEM engine (1 launch); scores and status words land at the caller's indices; an all-long batch is all tiled"""
    r = ctx(rna, 8, rna.ENGINE_AUTO)
    rs = np.random.RandomState(7500)
    lim = r.smem_max_n()
    seqs = [rand_seq(rs, n) for n in (100, lim + 1, 300, 0, 1500, lim, 64)]
    seqs[2] = seqs[2][:17] + b"X" + seqs[2][18:]
    seqs[4] = seqs[4][:900] + b"n" + seqs[4][901:]
    flat, offsets, lens32 = workloads.pack_batch(seqs)
    status = torch.full((len(seqs),), -7, dtype=torch.int32, device="cuda")
    scores = r.fold_batch(torch.from_numpy(flat).cuda(), torch.from_numpy(offsets).cuda(), lens32, status_out=status)
    torch.cuda.synchronize()
    assert r.last_launch_count() == 6
    want = np.array([oracle.nussinov_fast(s)["score"] if len(s) > 400 else oracle.nussinov(s) for s in seqs])
    assert want[2] == -1 and want[4] == -1
    assert (scores.cpu().numpy() == want).all()
    assert status.cpu().numpy().tolist() == [0, 0, 1, 0, 1, 0, 0]
    longs = [seqs[1], seqs[4]]
    flat, offsets, lens32 = workloads.pack_batch(longs)
    scores = r.fold_batch(torch.from_numpy(flat).cuda(), torch.from_numpy(offsets).cuda(), lens32)
    torch.cuda.synchronize()
    assert r.last_launch_count() == 5
    assert scores.cpu().numpy().tolist() == [want[1], -1]
    rs_ = ctx(rna, 8, rna.ENGINE_SMEM)
    with pytest.raises(rna.Rna4rError) as e:
        rs_.fold(dev_seq(seqs[1]))
    assert e.value.code == -3
    r9 = rna.Rna4r(9, 0)
    with pytest.raises(rna.Rna4rError) as e:
        r9.set_engine(rna.ENGINE_SMEM)
    assert e.value.code == -9
    r9.close()


@pytest.mark.parametrize("hi", [120, 330, 400, 470, 560])
def test_batches_of_every_cta_class(rna, hi):
    """the CTA size follows the longest sequence of the batch: 6, 8, 12 warps (four, three, two CTAs per SM) and 24"""
    r = ctx(rna, 8, rna.ENGINE_AUTO)
    seqs, _ = workloads.random_sequences(7700 + hi, 300, hi // 3, hi)
    seqs[0] = rand_seq(np.random.RandomState(hi), hi)
    flat, offsets, lens32 = workloads.pack_batch(seqs)
    scores = r.fold_batch(torch.from_numpy(flat).cuda(), torch.from_numpy(offsets).cuda(), lens32)
    torch.cuda.synchronize()
    assert r.last_launch_count() == 1
    want = np.array([oracle.nussinov_fast(x)["score"] for x in seqs])
    assert (scores.cpu().numpy() == want).all()


@pytest.mark.parametrize("q", [5, 8])
def test_random_batches_over_the_whole_length_range(rna, q):
    """lengths anywhere in 0..smem_max_n, mixed in one batch (the 24-warp class), several batches"""
    r = ctx(rna, q, rna.ENGINE_AUTO)
    lim = r.smem_max_n()
    for rep in range(3):
        seqs, _ = workloads.random_sequences(7800 + 10 * q + rep, 150, 0, lim)
        flat, offsets, lens32 = workloads.pack_batch(seqs)
        scores = r.fold_batch(torch.from_numpy(flat).cuda(), torch.from_numpy(offsets).cuda(), lens32)
        torch.cuda.synchronize()
        assert r.last_launch_count() == 1
        want = np.array([oracle.nussinov_fast(x, threads=2)["score"] for x in seqs])
        assert (scores.cpu().numpy() == want).all(), (q, rep)


def test_host_batch_and_repeat(rna):
    r = ctx(rna, 8, rna.ENGINE_AUTO)
    seqs, _ = workloads.random_sequences(7600, 200, 0, 500)
    flat, offsets, lens32 = workloads.pack_batch(seqs)
    want = np.array([oracle.nussinov(x) for x in seqs])
    for _ in range(3):
        got = r.fold_batch_host(flat, lens32)
        assert (got == want).all()
