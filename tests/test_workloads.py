"""Host logic of the workload table (CPU): BASELINE.json's configs by name and the shape-by-name grammar that gives every
table row under profiles/ a `bench.py --workload` command.  Data only -- none of the method's arithmetic lives there."""
import math

import pytest

from paper_1209_0296_b200 import workloads as W


def test_named_configs_are_baseline_jsons():
    c = W.configs()
    assert (c["cfg1"].dims, c["cfg1"].L, c["cfg1"].T) == (2, 64, 2.269)
    assert (c["cfg2_T2.269"].dims, c["cfg2_T2.269"].L) == (2, 8192)
    assert (c["cfg3"].dims, c["cfg3"].L) == (3, 512)
    assert (c["cfg4"].dims, c["cfg4"].L, c["cfg4"].two_S) == (3, 256, 2)
    w5 = c["cfg5_c0.20"]
    assert (w5.model, w5.J, w5.L) == (W.NE_HEATBATH, 0.0, 8192)
    assert abs(1.0 / (1.0 + math.exp(1.0 / w5.T)) - 0.20) < 1e-12          # reading D6: c = 1/(1+exp(1/T))
    seeds = [w.seed for w in {**c, **W.extras()}.values()]
    assert len(set(seeds)) == len(seeds)                                   # no two named workloads share a seed
    assert W.by_name("cfg3") == c["cfg3"] and W.by_name("mid2d_1024").L == 1024


@pytest.mark.parametrize("name,want", [
    ("ising2d_736", dict(dims=2, L=736, two_S=1, model=W.ISING, T=2.269)),
    ("ising3d_96", dict(dims=3, L=96, two_S=1, model=W.ISING, T=4.5115)),
    ("spin1_3d_64", dict(dims=3, L=64, two_S=2, model=W.ISING, T=3.0, h=0.01)),
    ("ea2d_1024", dict(dims=2, L=1024, model=W.EA, T=1.0)),
    ("ea3d_128", dict(dims=3, L=128, model=W.EA, T=1.1)),
    ("potts2d_q3_2048", dict(dims=2, L=2048, two_S=2, model=W.POTTS, T=1.0 / math.log(1.0 + math.sqrt(3.0)))),
    ("potts3d_q8_64", dict(dims=3, L=64, two_S=7, model=W.POTTS)),
    ("ne2d_c0.3_512", dict(dims=2, L=512, model=W.NE_HEATBATH, J=0.0, T=W.ne_temperature(0.3))),
])
def test_shape_grammar(name, want):
    w = W.by_name(name)
    assert w.name == name and w.N == w.L ** w.dims
    for k, v in want.items():
        assert getattr(w, k) == v, (k, getattr(w, k), v)
    assert W.by_name(name) == w                                            # deterministic, seed included
    assert w.create_args()["seed"] == w.seed


@pytest.mark.parametrize("name", ["ising4d_64", "potts2d_64", "ne3d_c0.3_64", "ne2d_64", "cfg9", "ising2d_", "ea2d_x"])
def test_unknown_names_are_refused(name):
    with pytest.raises(KeyError):
        W.by_name(name)
