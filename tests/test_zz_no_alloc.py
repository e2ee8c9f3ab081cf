"""-m gpu test of rna4r_fold_static (include/rna4r.h): the fold that allocates nothing and keeps its scratch in a static
device array of the library.  Its score is compared, bit for bit, with the existing rna4r_fold path (and the oracle) on
calls in a row that share the array -- a long fold, then a short one that finds the long one's leftovers, then a long one
again.  Collected last on purpose (the suite runs with pytest -x); it passes alone in a fresh process and after the others.
"""
import numpy as np
import pytest

import oracle

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def rna():
    if not torch.cuda.is_available():
        pytest.fail("these tests need a CUDA device (no CPU fallback exists)")
    import paper_1307_7820_b200 as pkg
    return pkg


def rand_seq(rs, n):
    return bytes(np.frombuffer(b"ACGU", dtype=np.uint8)[rs.randint(0, 4, size=n)])


def dev_seq(s: bytes):
    return torch.from_numpy(np.frombuffer(s, dtype=np.uint8).copy()).cuda()


@pytest.mark.parametrize("q", [8, 10, 4])
def test_static_fold_matches_the_workspace_fold_on_calls_in_a_row(rna, q):
    r = rna.Rna4r(q, 0)
    r.fold_static_setup()
    nmax = r.fold_static_max_n()
    assert nmax >= 1500                                   # the stated limit: 8 MiB of scratch (2239 bases at q = 8)
    rs = np.random.RandomState(7000 + q)
    score = torch.full((1,), -7, dtype=torch.int32, device="cuda")
    for n in (nmax, 37, 0, 700, nmax - 1, 1, 5 * 8 * q + 3):
        s = rand_seq(rs, n)
        d = dev_seq(s) if n else torch.empty(0, dtype=torch.uint8, device="cuda")
        want, _ = r.fold(d, n)                            # the existing path, caller-supplied workspace
        r.fold_static(d, score, n)
        torch.cuda.synchronize()
        assert int(score.item()) == int(want.item()), (q, n)
        if n <= 800:
            assert int(score.item()) == oracle.nussinov(s), (q, n)
    r.close()


def test_static_fold_two_calls_back_to_back_on_one_stream(rna):
    """no synchronisation between the two calls: stream order is the only ordering the shared array needs"""
    r = rna.Rna4r(8, 0)
    r.fold_static_setup()
    rs = np.random.RandomState(7100)
    sa, sb = rand_seq(rs, 1500), rand_seq(rs, 333)
    da, db = dev_seq(sa), dev_seq(sb)
    out = torch.zeros(2, dtype=torch.int32, device="cuda")
    for _ in range(3):
        r.fold_static(da, out[0:1])
        r.fold_static(db, out[1:2])
    torch.cuda.synchronize()
    wa, _ = r.fold(da)
    wb, _ = r.fold(db)
    torch.cuda.synchronize()
    assert out.cpu().tolist() == [int(wa.item()), int(wb.item())]
    assert int(wb.item()) == oracle.nussinov(sb)
    r.close()


def test_static_fold_rejects_what_does_not_fit_and_bad_arguments(rna):
    r = rna.Rna4r(8, 0)
    r.fold_static_setup()
    nmax = r.fold_static_max_n()
    score = torch.full((1,), -7, dtype=torch.int32, device="cuda")
    d = dev_seq(b"A" * 64)
    with pytest.raises(rna.Rna4rError) as e:
        r.fold_static(d, score, nmax + 1)                 # size check comes before anything is read or enqueued
    assert e.value.code == -3
    with pytest.raises(rna.Rna4rError) as e:
        r.fold_static(d, score, -1)
    assert e.value.code == -3
    assert r.lib.rna4r_fold_static(r.h, d.data_ptr(), 64, None, None) == -2
    torch.cuda.synchronize()
    assert int(score.item()) == -7                        # untouched by the rejected calls
    r.fold_static(dev_seq(b"ACGX" * 10), score)           # reading g4: not a base -> -1
    torch.cuda.synchronize()
    assert int(score.item()) == -1
    r.close()
    r12 = rna.Rna4r(12, 0)
    with pytest.raises(rna.Rna4rError) as e:
        r12.fold_static_setup()
    assert e.value.code == -9
    r12.close()
