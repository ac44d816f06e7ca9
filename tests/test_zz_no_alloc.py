"""cao_space_repair_noalloc: repair for callers that are not allowed to allocate device memory.

Who that is: code running inside an allocator's or memory pool's own callback, a plugin whose host lends it input and
output buffers plus a stream and nothing else, a process whose device memory another component reserved in full at
start-up, a loop that cannot afford the device-wide synchronisation a cudaMalloc may cause.  The normal cao_space_repair
asks such a caller for scratch it cannot get; this entry point uses one fixed array inside libcao.so instead (3 MiB,
at most 65,536 rows per call, shared by every call on the device).

What is checked: the results are bit-identical (integer work: the tolerance is zero, as in every repair test) to the
existing cao_space_repair path on the same rows, on calls made one after the other, because the array still holds the
previous call's worklists and keys when the next call starts -- a shorter batch after a longer one, an all-valid batch
after one full of invalid rows, then a longer one again.  The file sorts last on purpose: `pytest -x` stops at the
first failure, and this test must not hide the parity tests.  It builds its own spaces and needs no other test to have
run (nor minds if they have: the static array is touched by nothing else)."""
import numpy as np
import pytest

import workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def _space(make):
    import paper_2606_28372_b200 as cao
    sp = make()
    return sp, cao.Space.from_space(sp).build()


def _random_rows(sp, gs, rng, count, n_valid):
    """count in-domain rows, the first n_valid of them copies of valid rows (repair must be the identity there)."""
    rows = np.stack([rng.integers(0, m, size=count) for m in sp.m], axis=1).astype(np.uint8)
    if n_valid:
        valid = gs.rows().cpu().numpy()[:, :len(sp.m)]
        rows[:n_valid] = valid[rng.integers(0, valid.shape[0], size=n_valid)]
    return rows


def _both(gs, rows, probe):
    """(existing path, no-allocation path) -> two (rank, key) pairs of host arrays."""
    want_rank, want_key = gs.repair(rows, use_probe=probe)
    d_rows = gs.pack_rows(rows)
    c = d_rows.shape[0]
    # poison the outputs so that an entry the kernels never wrote cannot pass by accident
    rank = torch.full((c,), -7, dtype=torch.int32, device=gs.device)
    key = torch.full((c,), -7, dtype=torch.int64, device=gs.device)
    gs.repair_noalloc(d_rows, rank, key, use_probe=probe)
    torch.cuda.synchronize()
    return (want_rank.cpu().numpy(), want_key.cpu().numpy()), (rank.cpu().numpy(), key.cpu().numpy())


# configs[1]: 16-byte rows, most invalid rows end in the bitmap probes; configs[3]: 32-byte rows, 1.2e-4 valid, so nearly
# every invalid row goes through both worklists to the table scan -- the part of the scratch that carries state.
@pytest.mark.parametrize("make", [W.space_cfg1, W.space_cfg3], ids=["cfg1", "cfg3"])
def test_noalloc_matches_existing_path_on_consecutive_calls(make):
    sp, gs = _space(make)
    rng = np.random.default_rng(2606)
    batches = [_random_rows(sp, gs, rng, 700, 5),        # fills the worklists
               _random_rows(sp, gs, rng, 130, 3),        # shorter: the tail of the array still holds call 1's data
               _random_rows(sp, gs, rng, 64, 64),        # every row valid: both worklists must come out empty
               _random_rows(sp, gs, rng, 1500, 0)]       # longer again, ragged against the 128-candidate scan tile
    for probe in (True, False):
        for rows in batches:
            (want_rank, want_key), (rank, key) = _both(gs, rows, probe)
            assert np.array_equal(key, want_key)
            assert np.array_equal(rank, want_rank)
    # the same batch twice in a row gives the same answer twice
    (_, want_key), (_, key1) = _both(gs, batches[0], True)
    (_, _), (_, key2) = _both(gs, batches[0], True)
    assert np.array_equal(key1, want_key) and np.array_equal(key2, want_key)


def test_noalloc_single_output_and_limits():
    import paper_2606_28372_b200 as cao
    sp, gs = _space(W.space_cfg1)
    rng = np.random.default_rng(7)
    rows = _random_rows(sp, gs, rng, 257, 2)
    want_rank, want_key = gs.repair(rows)
    d_rows = gs.pack_rows(rows)
    rank = torch.empty(257, dtype=torch.int32, device=gs.device)
    gs.repair_noalloc(d_rows, rank_out=rank)                           # key output left out
    assert torch.equal(rank, want_rank)
    key = torch.empty(257, dtype=torch.int64, device=gs.device)
    gs.repair_noalloc(d_rows, key_out=key)                             # rank output left out
    assert torch.equal(key, want_key)
    # the largest batch the static array takes, then one row more
    cap = cao.Space.REPAIR_NOALLOC_MAX_ROWS
    big = gs.pack_rows(_random_rows(sp, gs, rng, cap + 1, 0))
    out = torch.empty(cap + 1, dtype=torch.int32, device=gs.device)
    with pytest.raises(cao.CaoError) as e:
        gs.repair_noalloc(big, rank_out=out)
    assert e.value.code == -3 and str(cap) in str(e.value)
    gs.repair_noalloc(big[:cap], rank_out=out)
    want_rank, _ = gs.repair(big[:cap])
    assert torch.equal(out[:cap], want_rank)
    # an empty batch is a no-op, and per-kernel timing (it creates CUDA events) is refused rather than silently allocating
    gs.repair_noalloc(big[:0], rank_out=out)
    cao.profile_enable(True)
    try:
        with pytest.raises(cao.CaoError) as e:
            gs.repair_noalloc(d_rows, rank_out=rank)
        assert e.value.code == -2
    finally:
        cao.profile_enable(False)
    gs.repair_noalloc(d_rows, rank_out=rank)
    assert torch.equal(rank, gs.repair(rows)[0])
