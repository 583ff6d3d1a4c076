"""arc_hash_blocks_static (the K1 entry point that allocates nothing: its scratch is a fixed __device__ array inside the
library) against the existing path, arc_hash_blocks, bit for bit - this is integer work - on calls made one after the
other, so that whatever a call leaves in the shared scratch is seen not to matter.  Collected last on purpose (the
suite runs with pytest -x).  Passes alone in a fresh process and after the other tests: it owns no state but the
scratch array, which every call rewrites before it reads it."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def arc():
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device")
    from paper_2606_21238_b200 import arc as A
    A.load_library()   # fails loudly if the extension is missing
    return A


def batch(rng, lens, base_shift):
    """Requests of the given token lengths packed back to back, starting base_shift tokens into the buffer (so that the
    first request sits at every 4-byte misalignment of the 16-byte bulk copies)."""
    offsets = np.zeros(len(lens) + 1, np.int64)
    offsets[0] = base_shift
    offsets[1:] = base_shift + np.cumsum(lens)
    tokens = rng.integers(0, 128000, size=int(offsets[-1]) + 5, dtype=np.int64).astype(np.int32)
    return torch.from_numpy(tokens).cuda(), offsets


def both_ways(arc, tokens, offsets, poison):
    n = int((np.diff(offsets) // 16).sum())
    want = arc.hash_blocks(tokens, offsets)
    got = torch.full((n,), poison, dtype=torch.int64, device="cuda")       # the caller's output buffer; nothing else is allocated
    arc.hash_blocks_static(tokens, offsets, got)
    torch.cuda.synchronize()
    return got.cpu().numpy(), want.cpu().numpy()


def test_static_scratch_entry_matches_arc_hash_blocks_on_calls_in_a_row(arc):
    rng = np.random.default_rng(20260621238)
    # blocks per request around the segment size (128) and its multiples, ragged tails, requests without a full block
    shapes = [
        [16 * b + t for b, t in [(1, 0), (127, 3), (128, 0), (129, 15), (0, 7), (257, 1), (640, 9), (0, 0), (33, 5), (1024, 0)]],
        [16 * b + t for b, t in [(3000, 11), (2, 2)]],                                       # one long request: 24 segments
        [int(x) for x in rng.integers(0, 16 * 300, size=200)],                               # many short ones
        [16 * b + t for b, t in [(129, 15), (128, 0), (1, 0)]],                              # small again: stale scratch beyond it
    ]
    for call, lens in enumerate(shapes):
        tokens, offsets = batch(rng, lens, base_shift=call % 4)
        got, want = both_ways(arc, tokens, offsets, poison=-1 - call)
        assert got.shape == want.shape and got.size > 0
        bad = np.flatnonzero(got != want)
        assert bad.size == 0, f"call {call}: {bad.size} of {got.size} keys differ, first at {bad[:8]}"
    # the same input twice in a row gives the same keys twice
    tokens, offsets = batch(rng, shapes[0], base_shift=1)
    a, want = both_ways(arc, tokens, offsets, poison=-7)
    b, _ = both_ways(arc, tokens, offsets, poison=-8)
    assert np.array_equal(a, want) and np.array_equal(b, want)


def test_static_scratch_entry_refuses_what_does_not_fit(arc):
    tokens = torch.zeros(64, dtype=torch.int32, device="cuda")
    out = torch.zeros(8, dtype=torch.int64, device="cuda")
    # more requests than the 4 KB argument holds
    with pytest.raises(arc.ArcError) as e:
        arc.hash_blocks_static(tokens, np.zeros(255 + 1, np.int64), out)
    assert e.value.code == -3 and "253" in str(e.value)
    # more segments than the fixed scratch holds: 64 requests x 65 segments (validated on the host before anything is touched)
    lens = np.full(64, 16 * (128 * 64 + 1), np.int64)
    offsets = np.concatenate([[0], np.cumsum(lens)])
    with pytest.raises(arc.ArcError) as e:
        arc.hash_blocks_static(tokens, offsets, out)
    assert e.value.code == -3 and "4096" in str(e.value)
    # an empty call and a call without any full block are fine and touch nothing
    arc.hash_blocks_static(tokens, np.zeros(1, np.int64), out)
    arc.hash_blocks_static(tokens, np.array([0, 15, 30], np.int64), out)
    torch.cuda.synchronize()
    assert int(out.abs().sum()) == 0
