"""-m gpu: the compact parity set that is also run under compute-sanitizer (memcheck / synccheck / racecheck;
SURVEY.md section 4 tier (vi)); profiles/r02_sanitizer.md holds the commands and their error counts:

    compute-sanitizer --tool <tool> python -m pytest tests/test_gpu_sanitize.py -m gpu -x -q

Small n (<= 3T), q = 4, 8, 10, full tables and one ragged batch on every engine, every result against the oracle."""
import numpy as np
import pytest

import oracle
import workloads

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("q", [4, 8, 10, 11])
def test_small_folds_and_one_batch(q):
    if not torch.cuda.is_available():
        pytest.fail("needs a CUDA device (no CPU fallback exists)")
    import paper_1307_7820_b200 as pkg
    r = pkg.Rna4r(q, 0)
    assert (r.table() == oracle.rtable(q)).all()
    T = 8 * q
    rs = np.random.RandomState(31 + q)
    for n in (q + 1, T + 3, 3 * T - 5):
        s = bytes(np.frombuffer(b"ACGU", dtype=np.uint8)[rs.randint(0, 4, size=n)])
        want_score, want = oracle.nussinov(s, want_table=True)
        score, tab = r.fold(torch.from_numpy(np.frombuffer(s, dtype=np.uint8).copy()).cuda(), table_dtype=pkg.TABLE_INT32)
        torch.cuda.synchronize()
        assert int(score.item()) == want_score and (tab.cpu().numpy() == want).all(), (q, n)
    seqs, _ = workloads.random_sequences(41 + q, 6, 0, 2 * T + 5)
    flat, offsets, lens = workloads.pack_batch(seqs)
    want = np.array([oracle.nussinov(x) for x in seqs])
    for eng in (pkg.ENGINE_AUTO, pkg.ENGINE_TILED):        # AUTO: the batch runs on the SMEM engine when q is in 4..8
        r.set_engine(eng)
        got = r.fold_batch(torch.from_numpy(flat).cuda(), torch.from_numpy(offsets).cuda(), lens)
        torch.cuda.synchronize()
        assert (got.cpu().numpy() == want).all(), (q, eng)
    if q <= 8:                                              # the SMEM engine's single fold with the table
        r.set_engine(pkg.ENGINE_SMEM)
        s = seqs[-1] if len(seqs[-1]) else b"ACGU" * 9
        want_score, want_tab = oracle.nussinov(s, want_table=True)
        score, tab = r.fold(torch.from_numpy(np.frombuffer(s, dtype=np.uint8).copy()).cuda(), table_dtype=pkg.TABLE_INT32)
        torch.cuda.synchronize()
        assert int(score.item()) == want_score and (tab.cpu().numpy() == want_tab).all()
    r.close()
