"""Parity of EVERY launch shape of BASELINE.json config 5 (subdomain side {4,8,16,32,64} x degree {1,2,3,4} x
fp32/fp64, the (P, B, T) sweep) against the oracle, element by element.

The mesh is reduced (a few subdomains per side instead of hundreds) but the subdomain shape is the config's, and
`grid_blocks` makes hz_partition choose the variant as if the partition had the full-size number of subdomains: the
kernel, tile, cluster size, threads per block and shared memory are those of the full 38 M-DOF mesh (asserted against
a full-size partition for the headline shape in test_gpu_full_size.py).  Covers the cluster kernel at p = 1, 2, 4 with
2..16 CTAs per subdomain, the 37 249- and 66 049-DOF subdomains, the streamed fallback and the packed small-subdomain
kernel (several 25..289-DOF subdomains per thread block).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from paper_2606_21695_b200 import hz  # noqa: E402
from paper_2606_21695_b200.inputs import make_config  # noqa: E402
from test_gpu_parity import check_case  # noqa: E402

FULL_N = {1: 6144, 2: 3072, 3: 2048, 4: 1536}     # BASELINE.json config 5: 6144/p elements per side
SHAPES = {}                                        # (p, s, prec) -> launch shape, printed by the last test


def reduced(p, s):
    nsub = max(3, 24 // s)      # 6x6 subdomains of 4x4 elements ... 3x3 subdomains of 64x64 elements
    return make_config(5, n=nsub * s, p=p, sub_elems=s), (FULL_N[p] // s) ** 2


@pytest.mark.parametrize("prec", [hz.HZ_F32, hz.HZ_F64])
@pytest.mark.parametrize("s", [4, 8, 16, 32, 64])
@pytest.mark.parametrize("p", [1, 2, 3, 4])
def test_config5_launch_shape_matches_the_oracle(p, s, prec):
    inp, l_full = reduced(p, s)
    g = check_case(inp, prec, 0, n_outer=2, n_wh=2 if s <= 16 else 1, flags=dict(grid_blocks=l_full))
    i = g["info"]
    assert i.dofs_per_sub == (s * p + 1) ** 2
    SHAPES[(p, s, "f32" if prec == hz.HZ_F32 else "f64")] = (i.dofs_per_thread, i.cluster_size, i.subs_per_block,
                                                             i.threads_per_block, i.smem_bytes)


@pytest.mark.parametrize("prec", [hz.HZ_F32, hz.HZ_F64])
@pytest.mark.parametrize("p,s", [(1, 4), (1, 8), (2, 4), (3, 4), (3, 8), (4, 4)])
def test_config5_one_dof_per_thread_variant(p, s, prec):
    # "Both threading variants" (BASELINE.json config 5, T = 1): the one-DOF-per-thread kernel on the
    # subdomain shapes that fit 1024 threads
    inp, l_full = reduced(p, s)
    g = check_case(inp, prec, 1, n_outer=2, n_wh=2, flags=dict(grid_blocks=l_full))
    assert g["info"].dofs_per_thread == 1


def test_print_the_launch_shapes():
    for k in sorted(SHAPES):
        print("config5 shape", k, "-> dofs/thread, CTAs/sub, subs/block, threads, smem:", SHAPES[k])
    kinds = {v[:2] for v in SHAPES.values()}
    if SHAPES:   # the sweep really went through clusters of several sizes and through the streamed fallback or none
        assert any(c > 1 for _, c in kinds)
