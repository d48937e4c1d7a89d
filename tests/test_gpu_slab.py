"""Slab decomposition of the time direction (include/lqcd.h "Slab decomposition")
checked on ONE GPU (-m gpu): R slabs live in R contexts of one process and run one after the other,
stage by stage; the halo exchange and the all-reduce between the stages are device copies / sums done
here by the test.  No rank ever waits for another, so this is not a stand-in for R GPUs -- it proves
that the kernels, the ghost layout, the boundary phases and the stage order reproduce the single-lattice
result of the CPU oracle.  The torch.distributed plumbing of the real multi-process path is covered on
CPU by tests/test_slab_dist.py (gloo, world size 2 and 3).
"""
import numpy as np
import pytest

import lattice_util as lu
import lqcd_inputs as gen

pytestmark = pytest.mark.gpu

SEED = gen.BASE_SEED
PH = np.exp(1j * np.pi * np.array([0.3, 0.0, 1.0, 0.5]))     # a complex phase on the time boundary
AP = gen.antiperiodic_t()
DIMS = (8, 8, 8, 16)
TOL = {0: 1e-13, 1: 1e-5}


@pytest.fixture()
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1209_5942_b200.binding as b
    yield b
    for c in range(1, 8):
        b.lqcd_select_context(c)
        try:
            b.lqcd_finalize()
        except b.LqcdError:
            pass
    b.lqcd_select_context(0)


class Slabs:
    """R virtual ranks: context r holds the slab of rank r."""

    def __init__(self, B, dims, phases, U, R, precision=0, recon=18):
        self.B, self.dims, self.R = B, dims, R
        self.V, self.S3 = lu.volume(dims), dims[0] * dims[1] * dims[2]
        self.nt = dims[3] // R
        self.g = []
        for r in range(R):
            B.lqcd_select_context(r)
            B.lqcd_slab_init(dims, phases, r, R)
            B.lqcd_set_format(precision, recon)
            B.lqcd_set_stream()
            lo, hi = r * self.nt * self.S3, (r + 1) * self.nt * self.S3
            self.g.append(B.upload_gauge(U[lo:hi]))
        for parity in (0, 1):                       # time-like links of slice t = -1, once
            h = B.lqcd_slab_gauge_halo(parity)
            for r in range(R):
                src = self.g[(r - 1) % R]
                self.g[r][h["ghost_bwd"]:h["ghost_bwd"] + h["bytes"]] = src[h["send_hi"]:h["send_hi"] + h["bytes"]]
        self.h = B.lqcd_slab_spinor_halo()

    def each(self):
        for r in range(self.R):
            self.B.lqcd_select_context(r)
            yield r

    def upload(self, x_half, parity):
        n = self.V // 2 // self.R
        return [self.B.upload_spinor(x_half[r * n:(r + 1) * n], parity) for r in self.each()]

    def alloc(self):
        return [self.B.alloc_spinor() for _ in self.each()]

    def download(self, f, parity):
        return np.concatenate([self.B.download_spinor(f[r], parity) for r in self.each()])

    def exchange(self, f):
        h, n, R = self.h, self.h["bytes"], self.R
        for r in range(R):
            f[r][h["ghost_fwd"]:h["ghost_fwd"] + n] = f[(r + 1) % R][h["send_lo"]:h["send_lo"] + n]
            f[r][h["ghost_bwd"]:h["ghost_bwd"] + n] = f[(r - 1) % R][h["send_hi"]:h["send_hi"] + n]


def _round(a, precision):
    return a if precision == 0 else a.astype(np.complex64).astype(np.complex128)


@pytest.mark.parametrize("R", [1, 2, 4, 8])
@pytest.mark.parametrize("split", [False, True])
@pytest.mark.parametrize("precision,recon", [(0, 18), (0, 12), (1, 18), (1, 12)])
def test_slab_dslash_matches_oracle(B, oracle_mod, R, split, precision, recon):
    kappa = 0.15
    U = gen.gauge_haar(DIMS, SEED)
    x = gen.spinor_gaussian(lu.volume(DIMS) // 2, SEED)
    S = Slabs(B, DIMS, PH, U, R, precision, recon)
    for parity in (0, 1):
        fin, fout = S.upload(x, 1 - parity), S.alloc()
        if split:      # interior before the ghosts exist, boundary after
            for r in S.each():
                B.lqcd_slab_dslash(S.g[r], fin[r], fout[r], parity, kappa, 1)
            S.exchange(fin)
            for r in S.each():
                B.lqcd_slab_dslash(S.g[r], fin[r], fout[r], parity, kappa, 2)
        else:
            S.exchange(fin)
            for r in S.each():
                B.lqcd_slab_dslash(S.g[r], fin[r], fout[r], parity, kappa, 0)
        got = S.download(fout, parity)
        want = oracle_mod.dslash_eo(DIMS, PH, _round(U, precision), _round(x, precision), parity, kappa)
        assert np.isfinite(got).all()
        assert lu.rel_err(got, want) <= TOL[precision], (R, parity)


@pytest.mark.parametrize("R", [2, 4])
@pytest.mark.parametrize("dagger", [0, 1])
@pytest.mark.parametrize("precision,recon", [(0, 18), (1, 12)])
def test_slab_mhat_matches_oracle(B, oracle_mod, R, dagger, precision, recon):
    kappa, mu = 0.15, 0.1
    U = gen.gauge_haar(DIMS, SEED)
    x = gen.spinor_gaussian(lu.volume(DIMS) // 2, SEED)
    S = Slabs(B, DIMS, AP, U, R, precision, recon)
    fin, tmp, fout = S.upload(x, 0), S.alloc(), S.alloc()
    S.exchange(fin)
    for r in S.each():
        B.lqcd_slab_mhat_stage(S.g[r], fin[r], tmp[r], fout[r], kappa, mu, dagger, 1, 0)
    S.exchange(tmp)
    for r in S.each():
        B.lqcd_slab_mhat_stage(S.g[r], fin[r], tmp[r], fout[r], kappa, mu, dagger, 2, 0)
    got = S.download(fout, 0)
    want = oracle_mod.mhat(DIMS, AP, _round(U, precision), _round(x, precision), kappa, mu, dagger)
    assert lu.rel_err(got, want) <= TOL[precision]


def _virtual_cg(B, S, fb, fx, kappa, mu, tol, maxit, split):
    """binding.slab_cg with the communication replaced by copies between the virtual ranks."""
    import torch
    for r in S.each():
        B.lqcd_slab_cg_begin(S.g[r], fb[r], fx[r], kappa, mu, tol)
    nbytes = B.lqcd_spinor_bytes()

    def sums():
        out = []
        for _ in S.each():
            out.append(B.device_bytes(B.lqcd_slab_sum_ptr(), 8).view(torch.float64))
        return out

    def allreduce():
        s = sums()
        tot = torch.stack([v.clone() for v in s]).sum(dim=0)
        for v in s:
            v.copy_(tot)

    def stage(k, part=0):
        for _ in S.each():
            B.lqcd_slab_cg_stage(k, part)

    def hop(k):
        f = []
        for _ in S.each():
            f.append(B.device_bytes(B.lqcd_slab_cg_halo_field(k), nbytes))
        if split:
            stage(k, 1)
            S.exchange(f)
            stage(k, 2)
        else:
            S.exchange(f)
            stage(k, 0)

    stage(0); allreduce(); stage(1)
    for it in range(maxit):
        hop(2); hop(3); stage(4); allreduce(); stage(5)
        hop(6); hop(7); stage(8); allreduce(); stage(9)
        flags = [B.lqcd_slab_cg_poll() for _ in S.each()]
        assert len(set(flags)) == 1, "the ranks disagree on convergence / iteration count"
        if flags[0][0]:
            break
    for k in (11, 12, 13, 14):
        hop(k)
    stage(15); allreduce(); stage(16)
    out = []
    for _ in S.each():
        st = B.lqcd_slab_cg_end(True)
        out.append((st,) + tuple(B.lqcd_cg_stats()))
    return out


@pytest.mark.parametrize("R,split", [(2, False), (2, True), (4, True)])
def test_slab_cg_matches_single_lattice_and_oracle(B, oracle_mod, R, split):
    kappa, mu, tol = 0.15, 0.1, 1e-10
    U = gen.gauge_haar(DIMS, SEED)
    b = gen.spinor_gaussian(lu.volume(DIMS) // 2, SEED, gen.STREAM_SOURCE)
    # the single-lattice solve of the same system
    B.lqcd_select_context(0)
    B.lqcd_init(DIMS, AP)
    B.lqcd_set_stream()
    g0, s0, x0 = B.upload_gauge(U), B.upload_spinor(b, 0), B.alloc_spinor()
    assert B.lqcd_cg_mdagm(g0, s0, x0, kappa, mu, tol, 500) == 0
    it0, _, _ = B.lqcd_cg_stats()
    xs0 = B.download_spinor(x0, 0)

    S = Slabs(B, DIMS, AP, U, R)
    fb, fx = S.upload(b, 0), S.alloc()
    stats = _virtual_cg(B, S, fb, fx, kappa, mu, tol, 500, split)
    assert len(set(stats)) == 1, "every rank must report the same status, iterations and residuals"
    st, iters, rr, rt = stats[0]
    assert st == 0 and abs(iters - it0) <= 1
    xs = S.download(fx, 0)
    assert np.isfinite(xs).all()
    assert lu.rel_err(oracle_mod.mdagm(DIMS, AP, U, xs, kappa, mu), b) <= 1.05 * tol      # reading G14 (i)
    assert abs(rt - lu.rel_err(oracle_mod.mdagm(DIMS, AP, U, xs, kappa, mu), b)) <= 1e-12
    assert lu.rel_err(xs, xs0) <= 1e-8


def test_slab_argument_checks(B):
    B.lqcd_select_context(1)
    for dims, rank, R in [((8, 8, 8, 12), 0, 8), ((8, 8, 8, 12), 0, 4), ((4, 4, 2, 8), 0, 2), ((8, 8, 8, 16), 2, 2)]:
        with pytest.raises(B.LqcdError):        # N_t/R not an integer / odd; slice not a multiple of 32; bad rank
            B.lqcd_slab_init(dims, AP, rank, R)
    B.lqcd_slab_init(DIMS, AP, 0, 2)
    B.lqcd_set_stream()
    assert B.lqcd_spinor_bytes() == (2048 + 2 * 256) * 192          # 8 slices + 2 ghost slices of 256 sites
    assert B.lqcd_gauge_bytes() == (2048 + 2 * 256) * 8 * 144
    h = B.lqcd_slab_spinor_halo()
    assert h == {"send_lo": 0, "send_hi": (2048 - 256) * 192, "ghost_fwd": 2048 * 192, "ghost_bwd": (2048 + 256) * 192,
                 "bytes": 256 * 192}
    g, s, o = B.alloc_gauge(), B.alloc_spinor(), B.alloc_spinor()
    for call in (lambda: B.lqcd_mtm(g, s, o, 0.15, 0.1, 0), lambda: B.lqcd_cg_mdagm(g, s, o, 0.15, 0.1, 1e-8, 10),
                 lambda: B.lqcd_plaquette(g), lambda: B.lqcd_slab_dslash(g, s, o, 0, 0.15, 3),
                 lambda: B.lqcd_slab_cg_stage(2, 0)):
        with pytest.raises(B.LqcdError):
            call()
    B.lqcd_select_context(0)
    with pytest.raises(B.LqcdError):
        B.lqcd_select_context(8)


@pytest.mark.parametrize("overlap", [False, True])
def test_binding_slab_cg_driver_single_rank(B, oracle_mod, overlap):
    """binding.slab_cg, the torch.distributed driver, with world = 1: the rank is its own neighbour
    (block copies instead of send/recv, no all-reduce), every stage, poll and the true residual run
    through the same code a multi-process job uses."""
    kappa, mu, tol = 0.15, 0.1, 1e-10
    U = gen.gauge_haar(DIMS, SEED)
    b = gen.spinor_gaussian(lu.volume(DIMS) // 2, SEED, gen.STREAM_SOURCE)
    B.lqcd_select_context(0)
    B.lqcd_slab_init(DIMS, AP, 0, 1)
    B.lqcd_set_stream()
    g = B.upload_gauge(U)
    B.slab_exchange_gauge(g, 0, 1)
    s, x = B.upload_spinor(b, 0), B.alloc_spinor()
    st = B.slab_cg(g, s, x, kappa, mu, tol, 500, 0, 1, overlap=overlap, check_every=3)
    iters, rr, rt = B.lqcd_cg_stats()
    xs = B.download_spinor(x, 0)
    assert st == 0 and 20 <= iters <= 60
    true_rel = lu.rel_err(oracle_mod.mdagm(DIMS, AP, U, xs, kappa, mu), b)
    assert true_rel <= 1.05 * tol and abs(rt - true_rel) <= 1e-12
    # maxit reached: status 1, x = last iterate
    x2 = B.alloc_spinor()
    assert B.slab_cg(g, s, x2, kappa, mu, 1e-30, 3, 0, 1, overlap=overlap) == 1
    assert B.lqcd_cg_stats()[0] == 3


def test_binding_slab_cg_driver_on_a_side_stream(B, oracle_mod):
    """The library on a side stream while torch's current stream is another one: the driver issues its copies /
    point-to-point operations and all-reduces on the LIBRARY's stream (binding._OnLibraryStream), so halos are
    ordered against the kernels; the result equals the run on the default stream bit for bit."""
    import torch
    kappa, mu, tol = 0.15, 0.1, 1e-10
    U = gen.gauge_haar(DIMS, SEED)
    b = gen.spinor_gaussian(lu.volume(DIMS) // 2, SEED, gen.STREAM_SOURCE)
    B.lqcd_select_context(0)
    out = []
    for side in (None, torch.cuda.Stream()):
        B.lqcd_slab_init(DIMS, AP, 0, 1)
        assert B.library_stream() is None
        if side is not None:
            B.lqcd_set_stream(side)
            assert B.library_stream() is side
            with torch.cuda.stream(side):
                g = B.upload_gauge(U)
                s, x = B.upload_spinor(b, 0), B.alloc_spinor()
            side.synchronize()
        else:
            B.lqcd_set_stream()
            g = B.upload_gauge(U)
            s, x = B.upload_spinor(b, 0), B.alloc_spinor()
        # called from the default stream either way
        assert torch.cuda.current_stream().cuda_stream != getattr(side, "cuda_stream", -1)
        B.slab_exchange_gauge(g, 0, 1)
        assert B.slab_cg(g, s, x, kappa, mu, tol, 500, 0, 1, overlap=True) == 0
        torch.cuda.synchronize()
        import contextlib
        with (torch.cuda.stream(side) if side is not None else contextlib.nullcontext()):
            out.append((B.download_spinor(x, 0), B.lqcd_cg_stats()))
    assert out[0][1] == out[1][1] and np.array_equal(out[0][0], out[1][0])
    assert lu.rel_err(oracle_mod.mdagm(DIMS, AP, U, out[1][0], kappa, mu), b) <= 1.05 * tol
    with pytest.raises(RuntimeError):
        B.check_same_stream(side.cuda_stream, torch.cuda.current_stream().cuda_stream)
    B.lqcd_slab_init(DIMS, AP, 0, 1)
    # after lqcd_slab_cg_begin the single-lattice three-step solver stays closed (include/lqcd.h)
    g, s, x = B.alloc_gauge(), B.alloc_spinor(), B.alloc_spinor()
    B.lqcd_slab_cg_begin(g, s, x, kappa, mu, tol)
    for call in (lambda: B.lqcd_cg_iterate(1), B.lqcd_cg_finish):
        with pytest.raises(B.LqcdError) as e:
            call()
        assert e.value.status == B.LQCD_BAD_ARG
    B.lqcd_select_context(0)
    B.lqcd_init((4, 4, 4, 4), AP)
