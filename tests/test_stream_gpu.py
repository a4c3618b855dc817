"""ChunkStream (copy / compute overlap over consecutive chunks) returns, chunk by chunk, what spd_search_host returns."""
import dataclasses

import numpy as np
import pytest
import torch

import gen

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1611_09704_b200 import build as B
    B.ensure_built()
    import paper_1611_09704_b200 as P
    P.lib()
    return P


@pytest.mark.parametrize("mode,nmax", [("sqrt", 32), ("linear", 16)])
def test_chunk_stream_equals_search_host(P, mode, nmax):
    from paper_1611_09704_b200.stream import ChunkStream
    base = gen.get_config(1)
    cap = 4096
    chunks = [torch.from_numpy(gen.make_array(dataclasses.replace(base, cid=base.cid + 100 * k))).pin_memory() for k in range(5)]
    cs = ChunkStream(base.n_dm, base.n_t, nmax, mode, base.threshold, capacity=cap, depth=2)
    got = cs.run(chunks)
    arena = torch.empty(P.search_host_arena_bytes(base.n_dm, base.n_t, nmax, cap), dtype=torch.uint8, device="cuda")
    h_out = torch.zeros((cap, 4), dtype=torch.int32).pin_memory()
    h_cnt = torch.zeros(1, dtype=torch.int64).pin_memory()
    counts = []
    for k, h in enumerate(chunks):
        total = P.spd_search_host(h, nmax, mode, base.threshold, h_out, h_cnt, None, arena)
        want = np.sort(h_out[:total].numpy().view(P.CAND_DTYPE).reshape(-1), order=["dm", "t"])
        rec, total2 = got[k]
        assert total2 == total and np.sort(rec, order=["dm", "t"]).tobytes() == want.tobytes()
        counts.append(total)
    assert len(set(counts)) > 1 and min(counts) > 0        # the chunks differ, and every one has detections


def test_chunk_stream_refuses_to_overrun_its_slots(P):
    from paper_1611_09704_b200.stream import ChunkStream
    cs = ChunkStream(4, 2048, 8, "sqrt", 5.0, capacity=64, depth=1)
    h = torch.zeros((4, 2048), dtype=torch.float32).pin_memory()
    h[0, 5] = 1.0
    t = cs.submit(h)
    with pytest.raises(P.SpdError):
        cs.submit(h)
    rec, total, st = cs.result(t)
    assert int(st["n"][0]) == 4 * 2048
    with pytest.raises(P.SpdError):
        cs.result(t)
