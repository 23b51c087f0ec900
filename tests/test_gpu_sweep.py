"""BASELINE.json configs[4] (the throughput sweep): parity of its shape classes.  For a spread of sweep points -- every
value of prefix, C, K, L_d and B appears, the largest point included -- one full-size layer-step runs through
pdllm_step on seeded device-side Gaussians and 4 sampled (b, h) are compared with the fp64 oracle (SURVEY 8(d):
"parity on 4 sampled (b,h) per point"): scores, chunk ids (the oracle's top-K of the GPU's scores: random data has no
planted gap), O and LSE at the R12 gates.  `python bench.py --mode sweep` does the same for every point while timing."""
import pytest
import torch

import bench
from paper_2606_10537_b200 import workloads as W

pytestmark = pytest.mark.gpu

POINTS = [  # (prefix, C, K, L_d, B)
    (8192, 512, 2, 64, 1), (8192, 1024, 8, 256, 8), (16384, 512, 16, 512, 1), (16384, 1024, 4, 64, 8),
    (32768, 512, 8, 256, 1), (32768, 512, 16, 512, 8), (32768, 1024, 16, 512, 8), (32768, 1024, 2, 256, 1),
]


@pytest.mark.parametrize("pt", POINTS)
def test_sweep_point_sampled_parity(pt):
    from paper_2606_10537_b200 import binding as B
    B.lib()
    prefix, C, K, L_d, Bn = pt
    w = W.Workload("sweep", B=Bn, H=32, H_kv=32, d=128, N=prefix // C, C=C, K=K, keep=1.0, L_q=64, L_d=L_d, alpha=0.0,
                   unit_logits=False, seed=0)
    g = torch.Generator(device="cuda").manual_seed(20260615 + sum(pt))
    rnd = lambda *s: torch.randn(*s, generator=g, device="cuda", dtype=torch.float32).to(torch.bfloat16)
    shape = B.Shape.of(w)
    t = dict(Q=rnd(Bn, 32, w.L, 128), Kc=rnd(Bn, 32, w.N, C + 1, 128), Vc=rnd(Bn, 32, w.N, C + 1, 128),
             Kd=rnd(Bn, 32, w.L, 128), Vd=rnd(Bn, 32, w.L, 128), ws=B.alloc_workspace(shape, 0), out={})
    r = bench.sampled_parity(B, torch, w, shape, t)
    print(pt, r)
    assert r["ok"], r
