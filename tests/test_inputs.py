"""The seeded input generator: shapes, edge counts and match-set fractions of BASELINE.json's configs."""
import numpy as np

from sim3ba_inputs import CONFIGS, make_config, make_graph
from sim3ba_inputs.graphs import _make_edges


def test_edge_counts_match_baseline_configs():
    want = {1: (12, 2, 0), 2: (96, 0, 0), 3: (608, 20, 0), 4: (3036, 60, 0), 5: (6003, 0, 9)}
    for k, (E, inter, loops) in want.items():
        edges, kind, _ = _make_edges(CONFIGS[k])
        assert edges.shape == (E, 2) and (kind == 2).sum() == inter and (kind == 1).sum() == loops
        assert np.all(edges[:, 0] != edges[:, 1]) and edges.min() >= 0 and edges.max() < CONFIGS[k].n_kf
    assert [CONFIGS[k].n_kf for k in range(1, 6)] == [8, 32, 200, 1000, 2000]
    assert [CONFIGS[k].hw for k in range(1, 6)] == [3072, 196608, 196608, 49152, 196608]


def test_config1_is_deterministic_and_has_stated_fractions():
    a, b = make_config(1), make_config(1)
    for f in ("points", "conf", "edges", "match", "poses_gt", "poses_init"):
        assert np.array_equal(getattr(a, f), getattr(b, f))
    assert a.points.dtype == np.float32 and a.conf.dtype == np.float32 and a.match.dtype == np.int32
    frac = (a.match >= 0).mean(axis=1)
    assert np.allclose(frac, a.meta["valid_frac_target"], atol=2e-3)
    assert np.array_equal(a.poses_init[0], a.poses_gt[0]) and a.fixed_kf.tolist() == [0]
    assert np.allclose(np.linalg.norm(a.poses_init[:, 3:7], axis=1), 1.0)
    assert a.conf.min() > 0 and a.conf.max() < 1
    # about 10 % of the valid matches are outliers: they break the geometric run structure
    e = 0
    m = np.flatnonzero(a.match[e] >= 0)
    runs = np.diff(a.match[e][m].astype(np.int64)) == np.diff(m)
    assert 0.7 < runs.mean() < 0.9


def test_reduced_config3_has_two_gauges():
    g = make_graph(CONFIGS[3].scaled(kf_per_agent=6, height=12, width=16, n_inter=2))
    assert g.poses_init_raw is not None and g.n_kf == 12
    assert np.array_equal(g.poses_init_raw, g.poses_init)        # the start handed out is the raw one ...
    (e, moving, moving_is_i), = g.meta["gauge_sync_plan"]            # ... with the plan to synchronise it by the method
    assert g.edge_kind[e] == 2 and moving == list(range(6, 12))
    assert g.agent[g.edges[e, 0 if moving_is_i else 1]] == 1
    s_ratio = g.poses_init_raw[6:, 7] / g.poses_gt[6:, 7]
    assert 0.25 < s_ratio.mean() < 3.5


def test_config_params_are_the_preset_plus_the_damping_of_config5():
    from oracle import sim3_gn_oracle as orc
    from sim3ba_inputs import PRESETS, config_params
    for k in (1, 2, 3, 4):
        assert config_params(k) == PRESETS["config"] and config_params(k, "paper") == PRESETS["paper"]
    assert config_params(5) == dict(PRESETS["config"], lm_lambda=1e-4)
    assert orc.Params(**config_params(5)).lm_lambda == 1e-4 and orc.Params(**config_params(2)).lm_lambda == 0.0
