"""Host logic of the seeded input generators (no method arithmetic there to test)."""
import numpy as np
import torch

from paper_2607_02521_b200 import inputs


def test_bf16_rounding_matches_torch_rne():
    x = np.random.default_rng(0).standard_normal(100000).astype(np.float32) * 3
    x[:6] = [0.0, -0.0, 1.0, 1.00390625, 1.01171875, 65280.0]  # ties: to even
    got = inputs.f32_to_bf16_bits(x)
    want = torch.from_numpy(x).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    assert np.array_equal(got, want)
    back = inputs.bf16_bits_to_f64(got)
    assert np.array_equal(back, torch.from_numpy(x).to(torch.bfloat16).double().numpy())


def test_streams_are_seeded_prefix_stable_and_distributed_as_stated():
    a4 = inputs.make_activations(4, 96, seed=3)
    a9 = inputs.make_activations(9, 96, seed=3)
    assert np.array_equal(a4, a9[:4])                       # A(M) is a prefix of A(M')
    assert not np.array_equal(a4, inputs.make_activations(4, 96, seed=4))
    w1, w2 = inputs.make_weights(256, 512, seed=3)
    assert not np.array_equal(w1, w2)
    w1b, _ = inputs.make_weights(256, 512, seed=3)
    assert np.array_equal(w1, w1b)
    a = inputs.bf16_bits_to_f64(inputs.make_activations(512, 512, seed=1))
    w = inputs.bf16_bits_to_f64(w1)
    assert abs(a.mean()) < 0.01 and abs(a.std() - 1.0) < 0.01
    assert abs(w.mean()) < 0.001 and abs(w.std() - 0.02) < 0.0005


def test_shape_table_matches_baseline_json():
    import json, os, re
    bj = json.load(open(os.path.join(os.path.dirname(__file__), "..", "BASELINE.json")))
    for cfg, (name, (K, N, seed, Ms)) in zip(bj["configs"], inputs.SHAPES.items()):
        assert f"K={K}" in cfg and f"N={N}" in cfg, (cfg, name)
    assert sum(len(v[3]) for v in inputs.SHAPES.values()) == 22


def test_sample_rows_cover_every_tile_and_lane_quarter():
    r = inputs.sample_rows(300)
    assert r[0] == 0 and r[-1] == 299 and len(set(r)) == len(r)
    assert {0, 31, 32, 63, 64, 95, 96, 127, 128, 255, 256, 287, 288} <= set(r.tolist())
    assert inputs.sample_rows(1).tolist() == [0]
