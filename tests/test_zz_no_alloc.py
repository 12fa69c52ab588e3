"""The entry point that allocates nothing (include/tdr.h: tdr_dev_popctrl_noalloc) against the existing path (the driver's
k_popctrl through tdr_dev_popctrl), on two calls in a row and more.  Collected last on purpose (the suite runs with pytest -x).
Byte records: the comparison is bit-exact, as a sorted multiset (the existing path writes its copies in any order)."""
import numpy as np
import pytest

from paper_2506_00263_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _sorted_records(t):
    a = np.ascontiguousarray(t.cpu().numpy()).view(np.dtype((np.void, 48))).ravel()
    return np.sort(a)


def _fission_bank(n):
    """A real fission bank: the last generation's sites of a small cfg1 run on the GPU."""
    from paper_2506_00263_b200 import tdr
    P = tdr.Problem(W.cfg1(n=n, n_inactive=1, n_active=1))
    g = P.run()
    P.close()
    return g["bank"]


def test_no_alloc_population_control_matches_the_existing_path_call_after_call():
    import torch
    from paper_2506_00263_b200 import tdr
    bank_np = _fission_bank(30011)
    assert len(bank_np) > 20000
    bank = torch.from_numpy(bank_np.view(np.uint8).reshape(-1, 48).copy()).cuda()
    # three calls in a row on the shared static scratch: a full bank, then a shorter one with another ratio and generation
    # (whatever the first call left behind must not leak into it), then the first again (must reproduce itself bit for bit)
    cases = [(bank, 1.07, 3), (bank[:7001], 2.6, 4), (bank, 1.07, 3), (bank[:1], 5.5, 9), (bank[100:100 + 33], 0.4, 2)]
    first = None
    for k, (b, pr, gen) in enumerate(cases):
        cap = int(b.shape[0] * (pr + 1)) + 64
        ref, ref_total = tdr.dev_popctrl(b, cap, 12345, gen, pr)
        got, got_total = tdr.dev_popctrl(b, cap, 12345, gen, pr, noalloc=True)
        assert got_total == ref_total and got.shape == ref.shape, (k, got_total, ref_total)
        assert np.array_equal(_sorted_records(got), _sorted_records(ref)), k
        # the no-alloc variant also promises bank order: the copies of site i come before those of site i + 1
        pos = {bytes(r[:24]): i for i, r in enumerate(b.cpu().numpy())}
        idx = np.array([pos[bytes(r[:24])] for r in got.cpu().numpy()])
        assert np.all(np.diff(idx) >= 0), k
        if k == 0:
            first = got.cpu().numpy().copy()
        if k == 2:
            assert np.array_equal(got.cpu().numpy(), first)


def test_no_alloc_limits_and_overflow_are_reported():
    import torch
    from paper_2506_00263_b200 import tdr
    bank_np = _fission_bank(5003)
    bank = torch.from_numpy(bank_np.view(np.uint8).reshape(-1, 48).copy()).cuda()
    # beyond the static scratch: a clear TDR_EINVAL, nothing launched
    big = torch.zeros((524288 + 1, 48), dtype=torch.uint8, device="cuda")
    with pytest.raises(tdr.TdrError) as e:
        tdr.dev_popctrl(big, 16, 1, 1, 1.0, noalloc=True)
    assert e.value.code == -1 and "TDR_NOALLOC_MAX_SITES" in str(e.value)
    # an output array that is too small: the total is still reported, only next_cap sites are written
    ref, ref_total = tdr.dev_popctrl(bank, 10 * len(bank_np), 7, 2, 1.5)
    got, got_total = tdr.dev_popctrl(bank, 100, 7, 2, 1.5, noalloc=True)
    assert got_total == ref_total > 100 and got.shape[0] == 100
    full, _ = tdr.dev_popctrl(bank, 10 * len(bank_np), 7, 2, 1.5, noalloc=True)
    assert np.array_equal(got.cpu().numpy(), full[:100].cpu().numpy())
    # an empty bank
    got, total = tdr.dev_popctrl(bank[:0], 8, 7, 2, 1.5, noalloc=True)
    assert total == 0 and got.shape[0] == 0
    torch.cuda.synchronize()
