"""The seeded generators: deterministic, right shapes/dtypes, and shaped like the configs say."""
import numpy as np
import torch

from paper_2411_07321_b200 import workloads as W


def test_rng_is_counter_based_and_deterministic():
    i = torch.arange(1000, dtype=torch.int64)
    a = W.rng_uniform(1, 2, i)
    b = W.rng_uniform(1, 2, i[500:])
    assert torch.equal(a[500:], b)
    assert not torch.equal(a, W.rng_uniform(1, 3, i)) and not torch.equal(a, W.rng_uniform(2, 2, i))
    assert float(a.min()) >= 0.0 and float(a.max()) < 1.0
    n = W.rng_normal(3, 4, torch.arange(200000, dtype=torch.int64))
    assert abs(float(n.mean())) < 0.01 and abs(float(n.var()) - 1.0) < 0.02


def test_tiny_config_shapes_and_chunk_independence():
    cfg = W.scaled(W.CONFIGS["tiny"], 30000)
    a = W.generate(cfg, chunk=1 << 22)
    b = W.generate(cfg, chunk=7001)
    for x, y in zip(a.numpy(), b.numpy()):
        assert np.array_equal(x, y)
    assert a.u.dtype == torch.float32 and a.vis.dtype == torch.complex64 and a.weight.dtype == torch.float32
    assert a.M == 30000 and torch.all(a.weight == 1.0)
    assert cfg.n_bl == 120 and abs(cfg.dl * cfg.N - 0.2) < 1e-15
    pa = W.plan_args(cfg, a)
    assert pa["w_max"] > pa["w_min"] and pa["N"] == 256 and pa["Nw"] == 8 and pa["support"] == 7


def test_config_table_matches_baseline_json():
    c = W.CONFIGS
    assert [c[k].M for k in ("tiny", "10M", "100M", "500M", "hotspot")] == [10**5, 10**7, 10**8, 5 * 10**8, 10**9]
    assert [c[k].N for k in ("tiny", "10M", "100M", "500M", "hotspot")] == [256, 2048, 4096, 8192, 16384]
    assert [c[k].Nw for k in ("tiny", "10M", "100M", "500M", "hotspot")] == [8, 32, 64, 32, 16]
    assert [c[k].dtype for k in ("tiny", "10M", "100M", "500M", "hotspot")] == ["c128", "c64", "c128", "c64", "c64"]
    assert c["hotspot"].support == 9 and c["hotspot"].sigma == 1.3 and c["hotspot"].hotspot_frac == 0.7
    for k in c:
        assert c[k].n_times * c[k].n_bl * c[k].n_ch >= c[k].M
    assert len(c["100M"].freqs_hz) == 8 and c["100M"].freqs_hz[0] == 120e6 and c["100M"].freqs_hz[-1] == 168e6


def test_hotspot_recipe_concentrates_the_core():
    cfg = W.scaled(W.CONFIGS["hotspot"], 50000)
    v = W.generate(cfg)
    r = torch.sqrt(v.u.double() ** 2 + v.v.double() ** 2)
    frac = float((r < 200.0).double().mean())
    assert 0.68 < frac < 0.80
    w = v.weight
    assert float(w.min()) >= 0.5 and float(w.max()) <= 1.0
