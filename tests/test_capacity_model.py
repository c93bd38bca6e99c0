"""NEXT-3: the D-instance capacity model (Eq. 11-14).  CPU only.

Oracle pins (oracle_capacity / oracle_pd_ratio against things other than themselves):
  C1  exact-fraction hand evaluation of Eq. 11-13 with round numbers (both the capacity-bound and the
      bandwidth-bound branch of the min)
  C2  Eq. 14 with the paper's own printed measurements: Table I (tests/golden/table1_tp_td.json,
      PAPER.md:84-92) gives T_p and per-step T_d on the same model the paper validates on; at the
      validation workload ISL/OSL = 1000/150 the ratio computed from the bracketing
      Table I rows brackets the printed optimum 4.58.  A transposed t_p / t_d, a
      dropped OSL or an inverted ratio misses the bracket by an order of magnitude.
  C3  balance identity: at R = n_p / n_d the production rate n_p / t_p equals the consumption rate
      n_d * cc_d / (t_d * OSL) (PAPER.md:219-223 in words)
Library (host entry points of libkvpool.so) == oracle, and its argument checks.
"""
import json
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle
import paper_2511_20982_b200 as kv
from paper_2511_20982_b200 import binding as B

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def test_c1_hand_values():
    # capacity-bound: (80 - 8) GB x 2 - 70 GB = 74 GB; V_BW = 0.05 s x 0.8 x 2 x 3350 GB/s = 268 GB
    v_mem, v_bw, cc = oracle.capacity(80e9, 8e9, 70e9, 2, 3350e9, 0.8, 0.05, 1000, 150, 327680)
    assert v_mem == 74e9 and abs(v_bw - 268e9) < 1.0
    assert abs(cc - float(Fraction(74 * 10**9, (1000 + 75) * 327680))) < 1e-9
    # bandwidth-bound: TPOT SLO of 5 ms -> V_BW = 26.8 GB < 74 GB
    v_mem, v_bw, cc = oracle.capacity(80e9, 8e9, 70e9, 2, 3350e9, 0.8, 0.005, 1000, 150, 327680)
    assert abs(cc - float(Fraction(268 * 10**8, (1000 + 75) * 327680))) < 1e-9
    # the model does not fit
    assert oracle.capacity(80e9, 8e9, 200e9, 2, 3350e9, 0.8, 0.05, 1000, 150, 327680)[2] == 0.0


def _interp(x, xs, ys):
    return float(np.interp(x, xs, ys))


def test_c2_table1_brackets_the_printed_optimum():
    with open(os.path.join(GOLDEN, "table1_tp_td.json")) as f:
        t = json.load(f)
    seq = t["seq_len"]
    isl, osl = 1000, 150
    t_p = _interp(isl, seq, t["T_p_ms"]) * 1e-3                       # one prefill of ISL tokens
    ratios = []
    for cc in ("200", "248"):                                         # Table I's two highest concurrencies
        t_d = _interp(isl + osl / 2, seq, t["T_d_ms"][cc]) * 1e-3     # average resident length ISL + OSL/2 (Eq. 13)
        ratios.append(oracle.pd_ratio(float(cc), t_p, t_d, osl))
    assert min(ratios) < t["printed_optimum_1000_150"] < max(ratios), ratios
    assert 4.0 < min(ratios) and max(ratios) < 5.5


def test_c3_balance_identity():
    cc_d, t_p, t_d, osl = 207.0, 0.166, 0.05, 150.0
    R = oracle.pd_ratio(cc_d, t_p, t_d, osl)
    n_d = 3.0
    n_p = R * n_d
    assert abs(n_p / t_p - n_d * cc_d / (t_d * osl)) < 1e-9 * (n_p / t_p)


def test_library_matches_oracle():
    rng = np.random.default_rng(5)
    for _ in range(200):
        a = dict(m_gpu=rng.uniform(40e9, 200e9), m_reserved=rng.uniform(0, 20e9), m_model=rng.uniform(1e9, 300e9),
                 tp=int(rng.integers(1, 9)), bw=rng.uniform(1e12, 8e12), alpha=rng.uniform(0.3, 1.0),
                 t_d_slo=rng.uniform(0.005, 0.2), isl=float(rng.integers(0, 32768)), osl=float(rng.integers(1, 4096)),
                 m_token=float(rng.choice([131072, 327680, 163840, 4096])))
        got = B.kv_capacity(**a)
        want = oracle.capacity(a["m_gpu"], a["m_reserved"], a["m_model"], a["tp"], a["bw"], a["alpha"], a["t_d_slo"],
                               a["isl"], a["osl"], a["m_token"])
        assert np.allclose([got["v_mem"], got["v_bw"], got["cc_d"]], want, rtol=1e-14, atol=0)
        assert got["bandwidth_bound"] == (want[1] < want[0])
        if want[2] > 0:
            t_p, t_d = rng.uniform(0.01, 1.0), rng.uniform(0.005, 0.2)
            assert np.isclose(B.kv_optimal_pd_ratio(want[2], t_p, t_d, a["osl"]),
                              oracle.pd_ratio(want[2], t_p, t_d, a["osl"]), rtol=1e-14)


def test_library_argument_checks():
    ok = dict(m_gpu=180e9, m_reserved=8e9, m_model=70e9, tp=1, bw=7.7e12, alpha=0.9, t_d_slo=0.05, isl=1000.0,
              osl=150.0, m_token=327680.0)
    assert B.kv_capacity(**ok)["cc_d"] > 0
    for bad in [dict(tp=0), dict(alpha=0.0), dict(alpha=2.0), dict(osl=0.0), dict(m_token=0.0), dict(bw=-1.0),
                dict(t_d_slo=float("nan")), dict(isl=-1.0)]:
        with pytest.raises(B.KVError) as e:
            B.kv_capacity(**{**ok, **bad})
        assert e.value.status == B.KV_ERR_INVALID
    for bad in [(0.0, 1.0, 1.0, 1.0), (1.0, 0.0, 1.0, 1.0), (1.0, 1.0, -1.0, 1.0), (1.0, 1.0, 1.0, 0.0)]:
        with pytest.raises(B.KVError):
            B.kv_optimal_pd_ratio(*bad)
    cfg = kv.PoolConfig(num_layers=32, num_q_heads=32, num_kv_heads=8, head_dim=128, num_blocks=8, max_requests=4,
                        max_blocks_per_request=4)
    assert B.kv_token_bytes(cfg) == 131072           # config 3, 131 072 B per token
    # an FP8 pool: codes + the two fp32 row scales per (layer, kv head) — M_token of Eq. 13 shrinks by 1.94
    cfg8 = kv.PoolConfig(**{**cfg.__dict__, "kv_dtype": B.KV_DTYPE_FP8_E4M3})
    assert B.kv_token_bytes(cfg8) == 32 * 8 * (2 * 128 + 8) == 67584
    assert B.kv_token_bytes(cfg8) * cfg8.block_size * cfg8.num_blocks == B.kv_pool_kv_bytes(cfg8)
