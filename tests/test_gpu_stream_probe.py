"""lqcd_stream_probe (-m gpu): the paper's buffer-copy micro-benchmark (Fig. 5) kept as
the library's HBM probe.  Its results have a plain definition (a copy; an XOR over words; an XOR over
seven planes), written out here with numpy on the same bytes: bit-exact is the bar.  Buffers sit between
guard regions, sizes cover the empty case, less than one tile, a ragged tail and several grid strides.
"""
import numpy as np
import pytest

import lqcd_inputs as gen

pytestmark = pytest.mark.gpu

GUARD = 4096
ELEM_BYTES = {0: 4, 1: 8, 2: 16, 3: 144, 4: 192}
# multiples of 16 * 7 * 9 * 12 = 12096 bytes are legal for every (elem, mode)
UNIT = 12096
SIZES = [0, UNIT, 37 * UNIT, 2551 * UNIT]   # 0 B, 12 KB, 447 KB, 30.9 MB (> 1184 CTAs x one tile for 16-byte elements)


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1209_5942_b200.binding as b
    b.lqcd_init((4, 4, 4, 4), gen.antiperiodic_t())
    b.lqcd_set_stream()
    yield b
    b.lqcd_finalize()


def _guarded(torch, payload_bytes, fill):
    buf = torch.full((payload_bytes + 2 * GUARD,), fill, dtype=torch.uint8, device="cuda")
    return buf, buf[GUARD:GUARD + payload_bytes]


def _random_bytes(nbytes, seed):
    return np.random.default_rng(seed).integers(0, 256, size=nbytes, dtype=np.uint8)


@pytest.mark.parametrize("nbytes", SIZES)
@pytest.mark.parametrize("elem", [0, 1, 2, 3, 4])
def test_copy_is_a_copy(B, elem, nbytes):
    import torch
    host = _random_bytes(nbytes, 11 + elem)
    sbuf, src = _guarded(torch, nbytes, 0x5A)
    dbuf, dst = _guarded(torch, nbytes, 0xA5)
    src.copy_(torch.from_numpy(host))
    B.lqcd_stream_probe(elem, B.LQCD_STREAM_COPY, src, dst, nbytes)
    torch.cuda.synchronize()
    assert np.array_equal(dst.cpu().numpy(), host)
    assert bool((dbuf[:GUARD] == 0xA5).all()) and bool((dbuf[GUARD + nbytes:] == 0xA5).all())
    assert np.array_equal(src.cpu().numpy(), host)


@pytest.mark.parametrize("nbytes", SIZES)
@pytest.mark.parametrize("elem", [0, 1, 2])
def test_read_returns_the_xor_of_all_words(B, elem, nbytes):
    import torch
    host = _random_bytes(nbytes, 23 + elem)
    _, src = _guarded(torch, nbytes, 0x5A)
    src.copy_(torch.from_numpy(host))
    out_bytes = 8 * B.LQCD_STREAM_PROBE_BLOCKS
    dbuf, dst = _guarded(torch, out_bytes, 0)
    B.lqcd_stream_probe(elem, B.LQCD_STREAM_READ, src, dst, nbytes)
    torch.cuda.synchronize()
    got = np.bitwise_xor.reduce(dst.cpu().numpy().view(np.uint64)) if nbytes else np.uint64(0)
    want = np.bitwise_xor.reduce(host.view(np.uint64)) if nbytes else np.uint64(0)
    assert got == want
    assert bool((dbuf[:GUARD] == 0).all()) and bool((dbuf[GUARD + out_bytes:] == 0).all())


@pytest.mark.parametrize("nbytes", SIZES)
@pytest.mark.parametrize("elem", [0, 1, 2])
def test_mix71_is_the_xor_of_seven_planes(B, elem, nbytes):
    import torch
    host = _random_bytes(nbytes, 37 + elem)
    _, src = _guarded(torch, nbytes, 0x5A)
    src.copy_(torch.from_numpy(host))
    dbuf, dst = _guarded(torch, nbytes // 7, 0xA5)
    B.lqcd_stream_probe(elem, B.LQCD_STREAM_MIX71, src, dst, nbytes)
    torch.cuda.synchronize()
    want = np.bitwise_xor.reduce(host.reshape(7, nbytes // 7), axis=0) if nbytes else host
    assert np.array_equal(dst.cpu().numpy(), want)
    assert bool((dbuf[:GUARD] == 0xA5).all()) and bool((dbuf[GUARD + nbytes // 7:] == 0xA5).all())


def test_bad_arguments(B):
    import torch
    a = torch.zeros(4096, dtype=torch.uint8, device="cuda")
    b = torch.zeros(4096, dtype=torch.uint8, device="cuda")
    for args in [(5, 0, a, b, 1024), (-1, 0, a, b, 1024), (2, 3, a, b, 1024),      # elem / mode out of range
                 (3, 1, a, b, 144), (4, 2, a, b, 192 * 7),                          # AoS elements: COPY only
                 (2, 0, a, b, 1000), (3, 0, a, b, 160), (4, 0, a, b, 144), (1, 2, a, b, 1024),   # sizes
                 (2, 0, a[8:], b, 1024), (2, 0, a, b[4:], 1024),                    # alignment
                 (2, 0, 0, b, 1024), (2, 0, a, 0, 1024)]:                           # null pointers
        with pytest.raises(B.LqcdError) as err:
            B.lqcd_stream_probe(*args)
        assert err.value.status == B.LQCD_BAD_ARG


def test_fp64_probe_counts_its_chains(B):
    """a = b = 1: every link adds 1, so thread t ends with sum_c (t + c + iters) = 8 t + 28 + 8 iters, exactly."""
    import torch
    n = B.LQCD_STREAM_PROBE_BLOCKS * 256
    for iters in (0, 1, 5, 1000):
        out = torch.full((n + 16,), -1.0, dtype=torch.float64, device="cuda")
        B.lqcd_fp64_probe(1.0, 1.0, iters, out)
        torch.cuda.synchronize()
        t = np.arange(n, dtype=np.float64)
        assert np.array_equal(out[:n].cpu().numpy(), 8 * t + 28 + 8 * iters)
        assert bool((out[n:] == -1.0).all())
    # a general (a, b): the chain against the same recurrence in numpy (fma vs a*x+b: one rounding apart per link)
    out = torch.empty(n, dtype=torch.float64, device="cuda")
    B.lqcd_fp64_probe(0.5, 0.25, 40, out)
    x = np.arange(n, dtype=np.float64)[:, None] + np.arange(8, dtype=np.float64)[None, :]
    for _ in range(40):
        x = x * 0.5 + 0.25
    assert np.allclose(out.cpu().numpy(), x.sum(axis=1), rtol=1e-14, atol=0)
    for bad in [(float("nan"), 1.0, 1, out), (1.0, float("inf"), 1, out), (1.0, 1.0, -1, out), (1.0, 1.0, 1, 0)]:
        with pytest.raises(B.LqcdError) as err:
            B.lqcd_fp64_probe(*bad)
        assert err.value.status == B.LQCD_BAD_ARG
