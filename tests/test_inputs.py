"""Pins for the seeded input generator (kf_inputs) -- SURVEY.md Appendix A / C."""
import numpy as np

from kf_inputs import gen, workloads
from conftest import load_golden


def _hex16(a):
    return [f"0x{int(x):04X}" for x in np.asarray(a).view(np.uint16)]


def test_splitmix_selfcheck():
    g = load_golden("generator_spots.json")
    got = [f"0x{int(x):016X}" for x in gen.hash64(0, np.arange(3))]
    assert got == g["hash_key0_idx0_2"]


def test_spot_values():
    g = load_golden("generator_spots.json")
    q = gen.gen_q(0, 0, 0, 32)
    assert _hex16(q[0, :4]) == g["q_l0_r0_step0_h0_d0_3"]
    assert q[0, :4].astype(np.float64).tolist() == g["q_l0_r0_step0_h0_d0_3_values"]
    assert _hex16(gen.gen_k(0, 0, [0], 8)[0, 0, :4]) == g["K_l0_r0_g0_t0_d0_3"]
    assert _hex16(gen.gen_v(0, 0, [4], 8)[1, 0, 124:]) == g["V_l0_r0_g1_t4_d124_127"]


def test_distribution_cfg1_K():
    g = load_golden("generator_spots.json")["cfg1_K_stats"]
    k = gen.gen_k(0, 0, np.arange(4096), 8).astype(np.float64)
    assert abs(k.mean() - g["mean"]) < 2e-4
    assert abs(k.std() - g["std"]) < 1e-4
    assert abs(np.abs(k).max() - g["max_abs"]) < 0.01
    assert np.abs(k).max() <= 4.88


def test_positional_statelessness():
    a = gen.gen_k(3, 7, np.arange(10, 20), 8)
    b = gen.gen_k(3, 7, [15], 8)
    assert np.array_equal(a[:, 5:6, :].view(np.uint16), b.view(np.uint16))
    # streams, layers, requests are independent
    assert not np.array_equal(gen.gen_k(0, 0, [0], 8), gen.gen_v(0, 0, [0], 8))
    assert not np.array_equal(gen.gen_k(0, 0, [0], 8), gen.gen_k(1, 0, [0], 8))
    assert not np.array_equal(gen.gen_k(0, 0, [0], 8), gen.gen_k(0, 1, [0], 8))


def test_cfg3_lengths():
    g = load_golden("appendix_c_routing.json")["cfg3"]
    lens = workloads.cfg3_lengths()
    assert lens == g["lengths"]
    assert sum(lens) == g["total_tokens"]
    assert sum(-(-s // 32768) for s in lens) == g["total_ranges"]
    assert min(lens) >= 1024 and max(lens) <= 204800


def test_cfg5_lengths():
    g = load_golden("appendix_c_routing.json")["cfg5"]
    raw = workloads.cfg5_lengths(crosser_every=10 ** 9)  # no crossers -> raw draw
    # request 0 is always a crosser for any crosser_every, restore the raw check from index 1 on
    assert raw[1:8] == g["raw_first8"][1:]
    lens = workloads.cfg5_lengths()
    assert [lens[r] for r in range(0, 128, 8)] == g["crosser_lengths"]
    assert sum(lens) == g["sum_len0"]
    assert sum(-(-s // 16384) for s in lens) == g["ranges_at_load"]
    # exactly one event per crosser at step 4*(r/8)
    for r in range(0, 128, 8):
        k = 4 * (r // 8)
        assert (lens[r] + k) % 16384 == 0


def test_workload_shapes():
    w = workloads.cfg1()
    assert (w.n_q_heads, w.n_kv_heads, w.range_tokens, w.n_partitions, w.contexts) == (32, 8, 2048, 2, [4096])
    # per-layer KV bytes per token = 2*H_kv*d*2B = 4096 for both model shapes
    assert w.kv_bytes_per_token() == 4096
    assert workloads.cfg4().kv_bytes_per_token() == 4096
    assert workloads.cfg4().max_ranges() == 32
    assert workloads.cfg2().max_ranges() == 1
    assert workloads.cfg3().max_ranges() == 6
    w5 = workloads.cfg5()
    assert w5.batch == 128 and w5.max_ranges() == 9 and w5.total_ranges() == 625


def test_fig10_workload_names_parse_to_the_papers_head_shapes():
    # PAPER.md:322 (Fig. 10): GQA Q32:KV8, Q48:KV8, Q64:KV8; MHA Q32:KV32, Q40:KV40, Q48:KV48; batch 8-128; seq 2K-32K
    from kf_inputs import workloads
    for hq, hkv in workloads.FIG10_HEADS:
        wl = workloads.by_name(f"fig10_q{hq}kv{hkv}_b16_s32k")
        assert (wl.n_q_heads, wl.n_kv_heads, wl.batch, wl.contexts[0]) == (hq, hkv, 16, 32768)
        assert wl.kv_bytes_per_token() == 2 * hkv * 128 * 2            # PAPER.md:234, per layer
        assert wl.max_ranges(1) == 4 and wl.slots_per_partition(1) == 16
    import pytest
    with pytest.raises((KeyError, AssertionError)):
        workloads.by_name("fig10_q33kv8_b16_s32k")
