"""Seeded input generator: shapes, distributions, and independence of the Z partition."""
import numpy as np
import torch

import qsgw_inputs as qi


def test_configs_match_baseline_json():
    import json, os
    base = json.load(open(os.path.join(os.path.dirname(os.path.dirname(__file__)), "BASELINE.json")))
    assert len(base["configs"]) == 5
    import re
    for text, name in zip(base["configs"], ["tiny", "small", "medium", "large", "xl"]):
        c = qi.CONFIGS[name]
        num = lambda key: int(re.search(key + r"=(?:o\*v=)?(\d+)", text).group(1))
        assert (num("N"), num("o"), num("v"), num("naux"), num("n_s")) == (c.n_mo, c.n_occ, c.n_virt, c.n_aux, c.n_pole)
        assert int(re.search(r"seed (\d+)", text).group(1)) == c.seed
        assert c.n_pole == c.n_ov
        m = re.search(r"s-block (\d+)", text)
        assert (int(m.group(1)) if m else 0) == c.s_block


def test_tiny_inputs_shapes_and_ranges():
    cfg = qi.CONFIGS["tiny"]
    inp = qi.make_inputs(cfg)
    assert inp.B.shape == (80, 24, 24) and inp.Z.shape == (95, 95)
    assert torch.equal(inp.B, inp.B.transpose(1, 2))
    e = inp.eps.numpy()
    assert np.all(np.diff(e[:5]) >= 0) and np.all(np.diff(e[5:]) >= 0)
    assert -1.5 <= e[:5].min() and e[:5].max() <= -0.2 and 0.05 <= e[5:].min() and e[5:].max() <= 5.0
    om = inp.Omega.numpy()
    assert np.all(np.diff(om) >= 0) and 0.2 <= om.min() and om.max() <= 6.0
    assert inp.occ.tolist() == [1.0] * 5 + [0.0] * 19
    off = inp.B.numpy()[:, np.triu_indices(24, 1)[0], np.triu_indices(24, 1)[1]]
    assert abs(off.std() - 0.1 / np.sqrt(2)) < 0.005           # reading #11: off-diagonal std 0.0707
    assert abs(inp.Z.numpy().std() * np.sqrt(cfg.n_pole) - 1.0) < 0.03


def test_deterministic_and_partition_independent():
    cfg = qi.custom_config(12, 4, 9, n_pole=700, seed=7)
    Z = qi.make_Z(cfg)
    assert torch.equal(Z, qi.make_Z(cfg))
    for s0, s1 in [(0, 1), (100, 300), (255, 257), (256, 512), (511, 700)]:
        assert torch.equal(qi.make_Z(cfg, s0, s1), Z[:, s0:s1])
    assert torch.equal(qi.make_B(cfg), qi.make_B(cfg))
    assert not torch.equal(qi.make_B(cfg), qi.make_B(qi.custom_config(12, 4, 9, n_pole=700, seed=8)))


def test_flop_model_matches_survey_table():
    f = qi.flop_model(qi.CONFIGS["xl"])
    assert abs(f["F1"] / 1.30e14 - 1) < 0.01 and abs(f["F2"] / 1.02e15 - 1) < 0.01
    assert abs(f["F2sym"] / 5.11e14 - 1) < 0.01 and abs(f["F3"] / 2.55e14 - 1) < 0.01
    assert abs(f["F_min"] / 8.96e14 - 1) < 0.01
