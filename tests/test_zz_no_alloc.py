"""lqcd_plaquette_static (include/lqcd.h): the average plaquette with its scratch -- the per-warp partial sums -- in a
file-scope device array instead of the context's cudaMalloc'ed buffer, for callers that may not allocate.  -m gpu.

The file sorts last on purpose: the suite runs with pytest -x, and a failure here must not hide another test.

Bar: the two entry points run the same plaquette kernel and differ in the order of the final sum over the partials
only, so they agree to a few ulp of an O(1) average: |difference| <= 1e-14, the bound tests/test_gpu_gauge.py puts on
lqcd_plaquette against the oracle in double (1e-6 in single, as there).
"""
import numpy as np
import pytest

import lqcd_inputs as gen

pytestmark = pytest.mark.gpu

AP = gen.antiperiodic_t()
SEED = gen.BASE_SEED


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1209_5942_b200.binding as b
    return b


def _static(B, g):
    import torch
    out = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    B.lqcd_plaquette_static(g, out)
    torch.cuda.synchronize()
    return float(out.item())


def test_two_calls_in_a_row_match_the_allocating_path(B, oracle_mod):
    """Two calls back to back, the second on a SMALLER lattice and another field, so that the array still holds the first
    call's partials (more of them than the second call uses) when the second call runs."""
    for dims, U in (((8, 8, 8, 16), gen.gauge_haar((8, 8, 8, 16), SEED)),
                    ((6, 4, 10, 4), gen.gauge_near_identity((6, 4, 10, 4), SEED + 1, 0.3))):
        B.lqcd_init(dims, AP)
        B.lqcd_set_format(0, 18)
        B.lqcd_set_stream()
        g = B.upload_gauge(U)
        p_static = _static(B, g)
        p_alloc = B.lqcd_plaquette(g)
        assert abs(p_static - p_alloc) <= 1e-14, (dims, p_static, p_alloc)
        assert abs(p_static - oracle_mod.plaquette(dims, U)) <= 1e-14
    # the same field twice: the second call reproduces the first bit for bit (fixed summation order)
    assert _static(B, g) == p_static


@pytest.mark.parametrize("precision,recon,tol", [(0, 12, 1e-14), (1, 18, 1e-6), (1, 12, 1e-6)])
def test_storage_variants(B, oracle_mod, precision, recon, tol):
    dims = (4, 6, 2, 8)
    U = gen.gauge_near_identity(dims, SEED, 0.3)
    B.lqcd_init(dims, AP)
    B.lqcd_set_format(precision, recon)
    B.lqcd_set_stream()
    g = B.upload_gauge(U)
    for _ in range(2):
        p_static = _static(B, g)
        assert abs(p_static - B.lqcd_plaquette(g)) <= 1e-14      # same kernel, same partials: sum order only
        assert abs(p_static - oracle_mod.plaquette(dims, U)) <= tol


def test_the_largest_lattice_the_array_holds_and_the_first_one_it_does_not(B):
    """32^3 x 64 (BASELINE config 5) needs exactly LQCD_PLAQUETTE_STATIC_MAX_PARTIALS partial sums.  The field is the unit
    field with a seeded perturbation written straight into the internal buffer: the plaquette kernel multiplies whatever
    3x3 matrices it is given, and the comparison is between the two entry points on the same buffer."""
    import torch
    dims = (32, 32, 32, 64)
    B.lqcd_init(dims, AP)
    B.lqcd_set_format(0, 18)
    B.lqcd_set_stream()
    V = int(np.prod(dims))
    canon = torch.zeros((V, 4, 3, 3), dtype=torch.complex128, device="cuda")
    canon[:, :, 0, 0] = canon[:, :, 1, 1] = canon[:, :, 2, 2] = 1.0
    noise = torch.randn((V, 4, 3, 3, 2), dtype=torch.float64, device="cuda", generator=torch.Generator("cuda").manual_seed(5))
    canon += 0.05 * torch.view_as_complex(noise)
    del noise
    g = B.alloc_gauge()
    B.lqcd_pack_gauge(canon, g)
    del canon
    for _ in range(2):
        p_static = _static(B, g)
        p_alloc = B.lqcd_plaquette(g)
        assert 0.5 < p_alloc < 1.5
        assert abs(p_static - p_alloc) <= 1e-14, (p_static, p_alloc)
    del g
    # 8 * ceil(V / 256) = 69632 > 65536: rejected with a message, nothing launched, the output untouched
    B.lqcd_init((64, 32, 32, 34), AP)
    B.lqcd_set_format(0, 18)
    B.lqcd_set_stream()
    out = torch.full((1,), -7.0, dtype=torch.float64, device="cuda")
    n0 = B.lqcd_launch_count()
    with pytest.raises(B.LqcdError) as ei:
        B.lqcd_plaquette_static(out, out)      # any non-null pointer: the size check comes first
    assert ei.value.status == -3 and "static scratch array holds 65536" in str(ei.value)
    assert B.lqcd_launch_count() == n0
    torch.cuda.synchronize()
    assert float(out.item()) == -7.0
    B.lqcd_init((4, 4, 4, 4), AP)              # leave a small context behind
