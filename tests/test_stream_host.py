"""Host logic of the chunked stream (no GPU): the time-axis plan of stream.time_chunks."""
import pytest

from paper_1611_09704_b200.stream import time_chunks


@pytest.mark.parametrize("n_t,nmax,align,k", [(4096, 32, 1, 4), (4096, 100, 1, 2), (4096, 64, 4, 3), (4096, 128, 8, 5), (1000, 1, 1, 3),
                                               (512, 512, 1, 2)])
def test_time_chunks_cover_every_start_sample_once(n_t, nmax, align, k):
    step = (n_t - nmax + 1) // align * align
    T = n_t + k * step
    plan = time_chunks(T, n_t, nmax, align)
    assert len(plan) == k + 1 and plan[0][0] == 0
    owner = [0] * T
    for i, (s, length, keep) in enumerate(plan):
        last = i == len(plan) - 1
        assert s % align == 0 and length == n_t and s + length <= T
        assert keep == (length if last else step)
        if not last:
            assert keep + nmax - 1 <= length                 # a kept start sample sees every width inside its chunk
            assert plan[i + 1][0] == s + keep
        for t in range(s, s + keep):
            owner[t] += 1
    assert owner == [1] * T


def test_time_chunks_ragged_tail_and_bad_arguments():
    plan = time_chunks(10000, 4096, 33)
    assert plan[-1][0] + plan[-1][1] == 10000 and plan[-1][2] == plan[-1][1] and plan[-1][1] < 4096
    assert time_chunks(100, 4096, 16) == [(0, 100, 100)]
    for bad in [(0, 10, 1, 1), (100, 10, 11, 1), (100, 10, 0, 1), (100, 10, 4, 0), (100, 10, 8, 4)]:
        with pytest.raises(ValueError):
            time_chunks(*bad)
