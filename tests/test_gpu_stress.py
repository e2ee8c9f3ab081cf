"""-m gpu stress tests of the flag / mbarrier protocol of the persistent fill kernel (SURVEY.md section 4 tier (vi)):
many back-to-back folds on two streams, every grid size from one CTA up, every result compared bit for bit with the
oracle's stored values.  A latent ordering bug would be timing dependent; these runs vary the timing."""
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


def dev(s: bytes):
    return torch.from_numpy(np.frombuffer(s, dtype=np.uint8).copy()).cuda()


def test_two_streams_back_to_back(rna):
    """cfg4 batch x 200 on one stream (tiled engine: the flag protocol; then the SMEM engine a user's AUTO call takes)
    while cfg3 x 50 runs on another (separate contexts and workspaces)."""
    seqs, lens = workloads.gc_rich_batch()
    want4 = np.loadtxt(os.path.join(GOLD, "cfg4_scores.txt"), dtype=np.int64, comments="#")[:, 2]
    flat, offsets, lens32 = workloads.pack_batch(seqs)
    s3 = workloads.single_config("cfg3")
    want3 = 2761                                   # tests/golden/cfg3_expected.txt
    ra, rb = rna.Rna4r(8, 0, rna.ENGINE_TILED), rna.Rna4r(8, 0)
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    fd, od, d3 = torch.from_numpy(flat).cuda(), torch.from_numpy(offsets).cuda(), dev(s3)
    ra.set_engine(rna.ENGINE_AUTO)                 # the AUTO workspace also holds the SMEM engine's arrays
    wsa = torch.empty(ra.workspace_bytes_batch(lens32), dtype=torch.uint8, device="cuda")
    ra.set_engine(rna.ENGINE_TILED)
    wsb = torch.empty(rb.workspace_bytes(len(s3)), dtype=torch.uint8, device="cuda")
    NA, NB = 200, 50
    outa = torch.full((NA, len(lens32)), -7, dtype=torch.int32, device="cuda")
    outb = torch.full((NB,), -7, dtype=torch.int32, device="cuda")
    torch.cuda.synchronize()
    ia = ib = 0
    while ia < NA or ib < NB:                      # interleave the enqueues so both streams stay busy
        for _ in range(4):
            if ia < NA:
                ra.fold_batch(fd, od, lens32, scores_out=outa[ia], workspace=wsa, stream=sa)
                ia += 1
        if ib < NB:
            rb.fold(d3, score_out=outb[ib:ib + 1], workspace=wsb, stream=sb)
            ib += 1
    torch.cuda.synchronize()
    got4 = outa.cpu().numpy()
    assert (got4 == want4[None, :]).all(), np.argwhere(got4 != want4[None, :])[:5]
    assert (outb.cpu().numpy() == want3).all()
    ra.set_engine(rna.ENGINE_AUTO)
    outa.fill_(-7)
    for ia in range(NA):
        ra.fold_batch(fd, od, lens32, scores_out=outa[ia], workspace=wsa, stream=sa)
        if ia % 8 == 0:
            rb.fold(d3, score_out=outb[ia // 8:ia // 8 + 1], workspace=wsb, stream=sb)
    torch.cuda.synchronize()
    assert ra.last_launch_count() == 1
    assert (outa.cpu().numpy() == want4[None, :]).all()
    assert (outb.cpu().numpy() == want3).all()
    ra.close()
    rb.close()


@pytest.mark.parametrize("q", [4, 8, 10, 11])
def test_every_grid_size(rna, q):
    """the task list is claimed in order and a claimed task only waits on earlier ones: any grid completes and
    gives the same table -- 1, 2, 3, 7 CTAs in all, then 1..3 CTAs per SM"""
    r = rna.Rna4r(q, 0, rna.ENGINE_TILED)
    T = 8 * q
    rs = np.random.RandomState(900 + q)
    s = bytes(np.frombuffer(b"ACGU", dtype=np.uint8)[rs.randint(0, 4, size=5 * T + 11)])
    want_score, want = oracle.nussinov(s, want_table=True)
    seqs, _ = workloads.random_sequences(910 + q, 24, 0, 4 * T)
    flat, offsets, lens = workloads.pack_batch(seqs)
    wantb = np.array([oracle.nussinov(x) for x in seqs])
    fd, od = torch.from_numpy(flat).cuda(), torch.from_numpy(offsets).cuda()
    for total, per_sm in ((1, 0), (2, 0), (3, 0), (7, 0), (0, 1), (0, 2), (0, 3), (0, 0)):
        r.set_max_blocks(total)
        r.set_max_blocks_per_sm(per_sm)
        for _ in range(3):
            score, tab = r.fold(dev(s), table_dtype=rna.TABLE_INT32)
            got = r.fold_batch(fd, od, lens)
            torch.cuda.synchronize()
            assert int(score.item()) == want_score, (q, total, per_sm)
            assert (tab.cpu().numpy() == want).all(), (q, total, per_sm)
            assert (got.cpu().numpy() == wantb).all(), (q, total, per_sm)
    r.close()


def test_mixed_folds_repeat(rna):
    """a few hundred folds over mixed n and q, single and batched, against the oracle"""
    rs = np.random.RandomState(4242)
    for q in (5, 8, 9):
        r = rna.Rna4r(q, 0)
        T = 8 * q
        for rep in range(40):
            n = int(rs.randint(0, 9 * T))
            s = bytes(np.frombuffer(b"ACGU", dtype=np.uint8)[rs.randint(0, 4, size=n)])
            want = oracle.nussinov_fast(s, threads=2)["score"] if n > 400 else oracle.nussinov(s)
            sc, _ = r.fold(dev(s) if n else torch.empty(0, dtype=torch.uint8, device="cuda"), n)
            torch.cuda.synchronize()
            assert int(sc.item()) == want, (q, n)
        seqs, _ = workloads.random_sequences(77 + q, 64, 0, 3 * T)
        flat, offsets, lens = workloads.pack_batch(seqs)
        wantb = np.array([oracle.nussinov(x) for x in seqs])
        fd, od = torch.from_numpy(flat).cuda(), torch.from_numpy(offsets).cuda()
        for rep in range(20):
            got = r.fold_batch(fd, od, lens)
            torch.cuda.synchronize()
            assert (got.cpu().numpy() == wantb).all(), (q, rep)
        r.close()


def test_status_words(rna):
    """device-detected errors: score -1 and a per-sequence status word; other sequences unaffected"""
    rs = np.random.RandomState(5)
    seqs = [bytes(np.frombuffer(b"ACGU", dtype=np.uint8)[rs.randint(0, 4, size=n)]) for n in (50, 200, 0, 64, 130, 77)]
    seqs[1] = seqs[1][:100] + b"X" + seqs[1][101:]
    flat, offsets, lens = workloads.pack_batch(seqs)
    bad_off = offsets.copy()
    bad_off[5] -= 3                                 # sequence 4 grows by... no: [4] ends 3 early, [5] starts 3 early
    for eng in (rna.ENGINE_TILED, rna.ENGINE_DIAG):
        r = rna.Rna4r(8, 0, eng)
        st = torch.full((len(seqs),), 99, dtype=torch.int32, device="cuda")
        got = r.fold_batch(torch.from_numpy(flat).cuda(), torch.from_numpy(offsets).cuda(), lens, status_out=st)
        torch.cuda.synchronize()
        want = np.array([oracle.nussinov(x) for x in seqs])
        assert want[1] == -1
        assert (got.cpu().numpy() == want).all()
        assert st.cpu().numpy().tolist() == [0, 1, 0, 0, 0, 0]
        got = r.fold_batch(torch.from_numpy(flat).cuda(), torch.from_numpy(bad_off).cuda(), lens, status_out=st)
        torch.cuda.synchronize()
        g = got.cpu().numpy()
        assert st.cpu().numpy().tolist() == [0, 1, 0, 0, 2, 2]
        assert g[4] == -1 and g[5] == -1 and (g[[0, 2, 3]] == want[[0, 2, 3]]).all()
        r.close()
