"""Host logic of the slab-fused sweep (no GPU): the launch order gf_fusion_schedule produces must be a valid
topological order of the sweep's dependencies -- BLACK on timeslice t after RED on t-1, t, t+1 (periodic) -- and
cover every (parity, timeslice) exactly once."""
import pytest

import paper_1209_4008_b200 as gfm


@pytest.mark.parametrize("Nt", [4, 6, 8, 10, 32, 64, 128])
@pytest.mark.parametrize("chunk", [1, 2, 3, 4, 5, 7, 200])
@pytest.mark.parametrize("backward", [False, True])
def test_schedule_is_valid(Nt, chunk, backward):
    sched = gfm.gf_fusion_schedule(Nt, chunk, backward)
    red_done, black_done = set(), set()
    for parity, a, b in sched:
        assert 0 <= a < b <= Nt
        for t in range(a, b):
            if parity == 0:
                assert t not in red_done
                red_done.add(t)
            else:
                assert t not in black_done
                for nb in ((t - 1) % Nt, t, (t + 1) % Nt):
                    assert nb in red_done, (Nt, chunk, backward, t, nb, sched)
                black_done.add(t)
    assert red_done == set(range(Nt)) and black_done == set(range(Nt))
    # RED chunks are at most `chunk` slices; the walk direction is as asked
    reds = [(a, b) for p, a, b in sched if p == 0]
    assert all(b - a <= chunk for a, b in reds)
    starts = [a for a, _ in reds]
    assert starts == sorted(starts, reverse=backward)


def test_schedule_argument_errors():
    lib = gfm.load_library()
    assert lib.gf_fusion_schedule(0, 1, 0, None, 0) == gfm.GF_EINVAL
    assert lib.gf_fusion_schedule(8, 0, 0, None, 0) == gfm.GF_EINVAL
    assert lib.gf_fusion_schedule(8, 2, 0, None, 5) == gfm.GF_EINVAL
