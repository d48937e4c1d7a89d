"""The multi-process plumbing of the slab decomposition on CPU (gloo, world size 2 and 3): the halo
exchange of binding.slab_exchange_blocks (which block goes to which neighbour's ghost, cyclically,
also when both neighbours are the same rank) and the all-reduce that makes every rank see the same
scalar.  The kernels that consume the ghosts are checked on the GPU in tests/test_gpu_slab.py."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

FIELD, SLICE = 64, 8      # bytes of the "field" and of one time slice in this toy layout
H = {"send_lo": 0, "send_hi": FIELD - SLICE, "ghost_fwd": FIELD, "ghost_bwd": FIELD + SLICE, "bytes": SLICE}


def _field(rank):
    """Rank r's field: byte i of its sites is 16 r + i // SLICE (slice index in the low nibble)."""
    buf = torch.full((FIELD + 2 * SLICE,), 255, dtype=torch.uint8)
    buf[:FIELD] = torch.arange(FIELD, dtype=torch.uint8) // SLICE + 16 * rank
    return buf


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import paper_1209_5942_b200.binding as B
    dist.init_process_group("gloo", rank=rank, world_size=world)
    buf = _field(rank)
    n = H["bytes"]
    reqs = B.slab_exchange_blocks(buf, [(H["send_lo"], n, "prev"), (H["send_hi"], n, "next")],
                                  [(H["ghost_fwd"], n, "next"), (H["ghost_bwd"], n, "prev")], rank, world)
    for r in reqs:
        r.wait()
    total = torch.tensor([float(rank + 1)], dtype=torch.float64)
    dist.all_reduce(total)
    out[rank] = (buf.numpy().copy(), float(total[0]))
    dist.destroy_process_group()


def _check(world, port):
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
    last = FIELD // SLICE - 1
    for rank in range(world):
        buf, total = out[rank]
        nxt, prv = (rank + 1) % world, (rank - 1) % world
        assert (buf[:FIELD] == _field(rank).numpy()[:FIELD]).all()                 # own sites untouched
        assert (buf[FIELD:FIELD + SLICE] == 16 * nxt + 0).all()                    # forward ghost = first slice of rank+1
        assert (buf[FIELD + SLICE:] == 16 * prv + last).all()                      # backward ghost = last slice of rank-1
        assert total == world * (world + 1) / 2


def test_halo_exchange_and_allreduce_gloo_world2():
    _check(2, 29531)      # prev == next: two sends to and two receives from the same peer


def test_halo_exchange_and_allreduce_gloo_world3():
    _check(3, 29533)


def test_single_rank_is_its_own_neighbour():
    sys.path.insert(0, ROOT)
    import paper_1209_5942_b200.binding as B
    buf = _field(0)
    n = H["bytes"]
    assert B.slab_exchange_blocks(buf, [(H["send_lo"], n, "prev"), (H["send_hi"], n, "next")],
                                  [(H["ghost_fwd"], n, "next"), (H["ghost_bwd"], n, "prev")], 0, 1) == []
    b = buf.numpy()
    assert (b[FIELD:FIELD + SLICE] == 0).all() and (b[FIELD + SLICE:] == FIELD // SLICE - 1).all()


def test_slab_host_logic_without_gpu():
    """Sizes, halo offsets and argument checks of the slab ABI need no device."""
    sys.path.insert(0, ROOT)
    import paper_1209_5942_b200.binding as B
    B.lqcd_select_context(3)
    try:
        B.lqcd_slab_init((8, 8, 8, 16), [1, 1, 1, -1], 1, 2)
        assert B.lqcd_spinor_bytes() == (2048 + 2 * 256) * 192
        assert B.lqcd_slab_spinor_halo()["ghost_bwd"] == (2048 + 256) * 192
        g0, g1 = B.lqcd_slab_gauge_halo(0), B.lqcd_slab_gauge_halo(1)
        groups = (2048 + 512) // 32
        assert g0["bytes"] == 256 * 144 and g0["send_hi"] == (3 * groups + (2048 - 256) // 32) * 32 * 144
        assert g1["ghost_bwd"] - g0["ghost_bwd"] == 4 * groups * 32 * 144
        for bad in [((8, 8, 8, 12), 0, 8), ((4, 4, 2, 8), 0, 2), ((8, 8, 8, 16), 2, 2)]:
            try:
                B.lqcd_slab_init(bad[0], [1, 1, 1, -1], bad[1], bad[2])
                raise AssertionError(f"lqcd_slab_init accepted {bad}")
            except B.LqcdError:
                pass
    finally:
        B.lqcd_select_context(0)


def test_slab_driver_refuses_two_different_streams():
    """binding.slab_cg / slab_exchange_* issue torch.distributed's operations on the library's stream and check
    it (binding.check_same_stream): NCCL orders against torch's CURRENT stream, the kernels run on the stream of
    lqcd_set_stream, and nothing else ties the two.  The rule itself needs no device."""
    sys.path.insert(0, ROOT)
    import pytest
    import paper_1209_5942_b200.binding as B
    B.check_same_stream(0, 0)                      # legacy default stream on both sides
    B.check_same_stream(0x7F00DEAD, 0x7F00DEAD)
    B.check_same_stream(None, 0)
    for lib, cur in ((0x7F00DEAD, 0), (0, 0x7F00DEAD), (0x7F00DEAD, 0x7F00BEEF)):
        with pytest.raises(RuntimeError, match="not the library's stream"):
            B.check_same_stream(lib, cur)
    # CPU tensors (the gloo tests above) are outside the rule: the guard is a no-op for them
    with B._OnLibraryStream(torch.zeros(4, dtype=torch.uint8)) as g:
        assert g.cm is None
    assert B.library_stream() is None or not torch.cuda.is_available()
