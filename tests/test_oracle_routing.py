"""Pins for oracle/routing.py (integer routing / slot / append-position model)."""
import pytest

from oracle.routing import RoutingError, RoutingModel
from kf_inputs import workloads
from conftest import load_golden


def test_fig5_scenario():
    # [0,T/2)->A0, [T/2,T)->A1; when the context grows beyond T a new entry
    # [T,...)->A2 is appended without modifying anything else.
    T = 16
    m = RoutingModel(n_partitions=3, range_tokens=T // 2, max_requests=1, max_ranges_per_request=4,
                     slots_per_partition=2)
    m.open_request(0, T)
    assert m.route[0] == [(0, 0), (1, 0)]
    before = list(m.route[0])
    ev = m.token_boundary()
    assert ev == [(0, 2, 2, 0)]
    assert m.route[0][:2] == before and m.route[0][2] == (2, 0)
    assert m.append_position(0) == (2, 0, 0)


def test_closed_form_at_load():
    # range number n = sum_{r'<r} J_r' + j  ->  (n mod P, n div P)
    P, R = 5, 8
    lens = [3, 8, 9, 40, 1, 17, 64]
    m = RoutingModel(P, R, len(lens), 8, 10)
    for r, n in enumerate(lens):
        m.open_request(r, n)
    n = 0
    for r, L in enumerate(lens):
        J = -(-L // R)
        assert m.n_ranges(r) == J
        for j in range(J):
            assert m.route[r][j] == (n % P, n // P)
            n += 1
    assert m.rr_cursor == n and sum(m.free_head) == n


def test_tiny_scenario_appendix_c():
    g = load_golden("appendix_c_routing.json")["tiny"]
    m = RoutingModel(g["P"], g["R"], 3, 8, 8)
    for r, n in enumerate(g["load_lens"]):
        m.open_request(r, n)
    assert [[list(x) for x in m.route[r]] for r in range(3)] == g["after_load"]["routes"]
    assert m.free_head == g["after_load"]["free_head"] and m.rr_cursor == g["after_load"]["cursor"]
    for st in g["steps"]:
        ev = m.token_boundary()
        assert [[r, p, s] for (r, _, p, s) in ev] == st["opens"]
        assert [list(m.append_position(r)) for r in range(3)] == st["append"]
        m.step_commit()
        assert m.len == st["lens_after"]
        assert m.free_head == st["free_head"] and m.rr_cursor == st["cursor"]


def test_invariants_random_walk():
    import random
    rnd = random.Random(5)
    P, R, B = 3, 4, 6
    m = RoutingModel(P, R, B, 16, 64)
    for r in range(B):
        m.open_request(r, rnd.randrange(0, 20))
    seen = {}
    for step in range(40):
        prev = [list(x) for x in m.route]
        prev_fh = list(m.free_head)
        m.token_boundary()
        for r in range(B):
            assert m.route[r][:len(prev[r])] == prev[r]          # entries never change once written
            p, s, off = m.append_position(r)
            assert 0 <= off < R and (p, s) == m.route[r][-1]     # appends go to the tail range only
            assert off == m.len[r] - (len(m.route[r]) - 1) * R
        assert all(a >= b for a, b in zip(m.free_head, prev_fh))  # monotone
        used = [ps for r in range(B) for ps in m.route[r]]
        assert len(used) == len(set(used))                         # no (p, slot) used twice
        assert sum(m.free_head) == sum(len(x) for x in m.route) == m.rr_cursor
        m.step_commit()


def test_cfg3_load():
    g = load_golden("appendix_c_routing.json")["cfg3"]
    w = workloads.cfg3()
    m = RoutingModel(w.n_partitions, w.range_tokens, w.batch, 8, 8)
    for r, S in enumerate(w.contexts):
        m.open_request(r, S - 1)      # S-1 resident, the S-th arrives at step 0 (SURVEY 8(d) state prep)
    m.token_boundary()
    assert m.free_head == g["slots_after_load"]
    assert [list(x) for x in m.route[2]] == g["request2_route"]
    assert sum(len(x) for x in m.route) == g["total_ranges"]


def test_cfg5_events():
    g = load_golden("appendix_c_routing.json")["cfg5"]
    w = workloads.cfg5()
    lens0 = w.extra["len_before_step0"]
    m = RoutingModel(w.n_partitions, w.range_tokens, w.batch, 9, 40)
    for r, n in enumerate(lens0):
        m.open_request(r, n)
    assert m.free_head == g["free_head_after_load"] and m.rr_cursor == g["ranges_at_load"]
    events = []
    for step in range(64):
        for (r, j, p, s) in m.token_boundary():
            events.append((step, r))
        m.step_commit()
    assert events == [(4 * i, 8 * i) for i in range(16)]
    assert m.free_head == g["free_head_final"] and m.rr_cursor == g["cursor_final"]
    assert [list(x) for x in m.route[0]] == g["request0_final_route"]
    assert [list(x) for x in m.route[120]] == g["request120_final_route"]


def test_close_and_lifo_reuse():
    m = RoutingModel(2, 4, 3, 4, 4)
    m.open_request(0, 8)   # (0,0),(1,0)
    m.open_request(1, 4)   # (0,1)
    m.close_request(0)     # free lists: p0:[0], p1:[0]
    assert m.len[0] == -1 and m.route[0] == []
    m.open_request(2, 8)   # cursor=3 -> p1 reuse slot 0 ; cursor=4 -> p0 reuse slot 0
    assert m.route[2] == [(1, 0), (0, 0)]
    assert m.free_head == [2, 1]
    with pytest.raises(RoutingError):
        m.open_request(1, 4)
    with pytest.raises(RoutingError):
        m.close_request(0)


def test_enospc():
    m = RoutingModel(1, 4, 1, 8, 2)
    m.open_request(0, 8)
    with pytest.raises(RoutingError):
        m.token_boundary()
    m2 = RoutingModel(2, 4, 1, 2, 8)
    m2.open_request(0, 8)
    with pytest.raises(RoutingError):
        m2.token_boundary()


def test_full_partition_is_passed_over():
    # reading 24, worked by hand: P = 2, 2 slots each, R = 4.  Only node 0 is active while request 0 loads 8 tokens:
    # both of its ranges land on node 0 -> (0,0),(0,1): node 0 is full.  Node 1 joins.  Request 1 (4 tokens): the
    # first active node after node 0 is node 1 -> (1,0).  Request 2 (4 tokens): the round-robin would return to node 0,
    # which has no free slot, so it is passed over -> (1,1).  Now everything is full: ENOSPC.
    m = RoutingModel(2, 4, 4, 4, 2)
    m.set_active([1, 0])
    m.open_request(0, 8)
    assert m.route[0] == [(0, 0), (0, 1)]
    m.set_active([1, 1])
    m.open_request(1, 4)
    assert m.route[1] == [(1, 0)]
    m.open_request(2, 4)
    assert m.route[2] == [(1, 1)]
    assert m.free_head == [2, 2] and m.rr_cursor == 4
    with pytest.raises(RoutingError):
        m.open_request(3, 1)


def test_request_waits_for_a_slot_and_resumes():
    # reading 24, worked by hand: P = 1, 3 slots, R = 4.  r0 holds 4 tokens in slot 0, r1 holds 8 in slots 1, 2.
    # Boundary: both tail ranges are full and no slot is left -> ENOSPC, nobody gets a range; the commit leaves both
    # where they are (nothing was appended).  r1 is closed: slots 1 then 2 go on the LIFO list.  Next boundary: r0 takes
    # slot 2 (top of the list), appends at offset 0 of it, commits to 5.  r2 opens with 1 token -> slot 1.
    m = RoutingModel(1, 4, 3, 4, 3)
    m.open_request(0, 4)
    m.open_request(1, 8)
    assert m.route == [[(0, 0)], [(0, 1), (0, 2)], []]
    for _ in range(2):                       # waiting does not move anything, however often it is re-tried
        with pytest.raises(RoutingError):
            m.token_boundary()
        assert m.last_events == []
        with pytest.raises(RoutingError):
            m.append_position(0)
        m.step_commit()
        assert m.len == [4, 8, -1] and m.rr_cursor == 3
    m.close_request(1)
    assert m.token_boundary() == [(0, 1, 0, 2)]
    assert m.append_position(0) == (0, 2, 0)
    m.step_commit()
    assert m.len == [5, -1, -1]
    m.open_request(2, 1)
    assert m.route[2] == [(0, 1)]
    # a boundary where one request finds a slot and a later one does not: the first still gets its range
    m2 = RoutingModel(1, 2, 2, 4, 3)
    m2.open_request(0, 2)
    m2.open_request(1, 2)                    # slots 0, 1 used, one left
    with pytest.raises(RoutingError):
        m2.token_boundary()
    assert m2.last_events == [(0, 1, 0, 2)] and m2.route[1] == [(0, 1)]
    m2.step_commit()
    assert m2.len == [3, 2]


def test_kv_byte_formula():
    # PAPER.md:234 C_total = sum_i 2*s_i*H_kv*d_h*L*2B; PAPER.md:35 sanity: Llama-3.1-8B, batch 64 x 4K
    # tokens = 32 GiB (128 KiB/token over 32 layers)
    per_token = 2 * 8 * 128 * 32 * 2
    assert per_token == 128 * 1024
    assert 64 * 4096 * per_token == 32 * 2 ** 30


# ---- active sets: scale-up / scale-down events (Fig. 5 at :173) -------------------------
def test_fig5_scale_up_appends_route_on_the_new_node_only():
    # Fig. 5 caption: [0,T/2) -> A0, [T/2,T) -> A1, then A2 is published and [T,...) -> A2; nothing else changes
    R = 8
    m = RoutingModel(3, R, 1, 4, 4)
    m.set_active([1, 1, 0])
    m.open_request(0, 2 * R)                         # T = 2R tokens after prefill
    assert m.route[0] == [(0, 0), (1, 0)]
    before = list(m.route[0])
    m.set_active([1, 1, 1])                          # the prewarmed node's route is published
    ev = m.token_boundary()                          # len % R == 0: the tail range is full -> a new range opens
    assert ev == [(0, 2, 2, 0)]
    assert m.route[0][:2] == before and m.route[0][2] == (2, 0)
    assert m.append_position(0) == (2, 0, 0)


def test_all_partitions_active_is_k_mod_p():
    import random
    rnd = random.Random(7)
    P, R = 5, 4
    m = RoutingModel(P, R, 6, 64, 64)
    k = 0
    for r in range(6):
        n = rnd.randrange(0, 40)
        m.open_request(r, n)
        for j in range(-(-n // R)):
            assert m.route[r][j][0] == k % P
            k += 1
    for _ in range(30):
        for (_, _, p, _) in m.token_boundary():
            assert p == k % P
            k += 1
        m.step_commit()
    assert m.rr_cursor == k


def test_scale_down_keeps_existing_ranges_and_starves_the_retired_node():
    P, R = 3, 4
    m = RoutingModel(P, R, 3, 32, 32)
    for r, n in enumerate([9, 4, 6]):
        m.open_request(r, n)
    frozen = [list(x) for x in m.route]
    m.set_active([1, 0, 1])                          # node 1 leaves the active set
    for _ in range(24):
        m.token_boundary()
        m.step_commit()
    for r in range(3):
        assert m.route[r][:len(frozen[r])] == frozen[r]              # entries never change once written
        assert all(p != 1 for (p, _) in m.route[r][len(frozen[r]):])  # no new range on the retired node
    st = m.partition_state()
    assert sum(st["tokens"]) == sum(m.len) and sum(st["tails"]) == 3 and st["active"] == [1, 0, 1]
    assert st["tails"][1] == 0                        # every tail has moved on since
    # bytes the policy sees: tokens x 2 * H_kv * d_h * L * 2 B
    assert st["tokens"][0] * 2 * 8 * 128 * 32 * 2 == st["tokens"][0] * 131072
    with pytest.raises(RoutingError):
        m.set_active([0, 0, 0])


def test_paused_requests_keep_routes_and_length():
    # continuous batching: a request that sits out steps ("r active", Algorithm 1 l.7) is frozen -- no range is
    # opened for it even at a range edge, its length does not move, it is not counted as a tail -- and resumes intact
    R = 4
    m = RoutingModel(2, R, 3, 8, 8)
    for r, n in enumerate([4, 3, 6]):             # request 0 sits exactly at a range edge
        m.open_request(r, n)
    m.set_active_requests([0, 1, 1])
    routes0 = list(m.route[0])
    for _ in range(5):
        ev = m.token_boundary()
        assert all(e[0] != 0 for e in ev)
        m.step_commit()
    assert m.len == [4, 8, 11] and m.route[0] == routes0
    st = m.partition_state()
    assert sum(st["tails"]) == 2 and sum(st["tokens"]) == 4 + 8 + 11
    m.set_active_requests(None)                   # resume: now the edge opens range 1 for request 0
    ev = m.token_boundary()
    assert [e[:2] for e in ev if e[0] == 0] == [(0, 1)]
    m.step_commit()
    assert m.len[0] == 5 and sum(m.partition_state()["tails"]) == 3


# ---- reading 28: Algorithm 1 l.16-17 taken literally -- a published route redirects ACTIVE TAILS at the next boundary ----
def test_fig5_with_a_cut_at_t_plus_k_worked_by_hand():
    # Fig. 5 continued: T = 16, R = 8, three nodes.  [0,8)->A0, [8,16)->A1, the boundary at len = 16 opens
    # [16,..)->A2.  Three tokens later (len = 19) node A2 is over its threshold: the policy publishes a route without
    # A2 and redirects its tails.  At the NEXT boundary the tail [16,19) is closed where it is
    # and [19,..) opens on the first active node after A2 = A0; nothing older changes (:240).
    m = RoutingModel(n_partitions=3, range_tokens=8, max_requests=1, max_ranges_per_request=6, slots_per_partition=3)
    m.open_request(0, 16)
    for _ in range(3):
        m.token_boundary()
        m.step_commit()
    assert m.len[0] == 19 and m.route[0] == [(0, 0), (1, 0), (2, 0)] and m.begin[0] == [0, 8, 16]
    m.set_active([1, 1, 0])
    m.redirect_tails([0, 0, 1])
    assert m.token_boundary() == [(0, 3, 0, 1)]                      # A0's slot 0 holds [0,8): bump allocator gives slot 1
    assert m.route[0] == [(0, 0), (1, 0), (2, 0), (0, 1)] and m.begin[0] == [0, 8, 16, 19]
    assert m.append_position(0) == (0, 1, 0)                         # token 19 is the first token of the new range
    assert [m.range_tokens_held(0, j) for j in range(4)] == [8, 8, 3, 0]
    assert m.locate(0, 18) == (2, 0, 2) and m.locate(0, 16) == (2, 0, 0) and m.locate(0, 15) == (1, 0, 7)
    m.step_commit()
    assert m.locate(0, 19) == (0, 1, 0)
    # the marks are consumed: nothing moves at the following boundaries until the new tail is FULL (8 tokens: 19..26)
    for n in range(20, 27):
        assert m.token_boundary() == []
        assert m.append_position(0) == (0, 1, n - 19)
        m.step_commit()
    assert m.len[0] == 27
    assert m.token_boundary() == [(0, 4, 1, 1)]                      # 27 - 19 = 8 = R: next active node after A0 is A1
    assert m.begin[0] == [0, 8, 16, 19, 27]
    st = m.partition_state()
    assert st["tokens"] == [8 + 8, 8 + 0, 3] and st["tails"] == [0, 1, 0]


def test_redirect_moves_only_tails_on_marked_nodes_and_only_nonempty_ones():
    m = RoutingModel(3, 4, 3, 6, 4)
    m.open_request(0, 5)      # ranges -> A0, A1: tail on A1 holds token 4
    m.open_request(1, 2)      # A2: tail on A2
    m.open_request(2, 4)      # A0: tail full -> the boundary opens a range anyway
    m.redirect_tails([0, 1, 0])
    ev = m.token_boundary()
    # request 0: tail on the marked node A1, one token in it -> cut at 5; request 1: not marked; request 2: ordinary fill
    assert [(r, j) for r, j, _, _ in ev] == [(0, 2), (2, 1)]
    assert m.begin[0] == [0, 4, 5] and m.begin[1] == [0] and m.begin[2] == [0, 4]
    # a tail that holds no token yet (opened at the previous boundary, nothing committed since) is not cut again;
    # request 1's tail on A2 holds two tokens and IS cut now that every node is marked
    m.redirect_tails([1, 1, 1])
    ev = m.token_boundary()
    assert [(r, j) for r, j, _, _ in ev] == [(1, 1)]
    assert m.begin[0] == [0, 4, 5] and m.begin[1] == [0, 2] and m.begin[2] == [0, 4]


def test_redirect_without_a_free_slot_is_not_carried_out():
    m = RoutingModel(2, 4, 2, 4, 1)
    m.open_request(0, 2)      # A0 slot 0
    m.open_request(1, 2)      # A1 slot 0: every slot is taken
    m.redirect_tails([1, 0])
    assert m.token_boundary() == []          # no error, the tail stays
    assert m.append_position(0) == (0, 0, 2)
    m.step_commit()
    assert m.len == [3, 3]


def test_redirect_invariants_random_walk():
    import random
    rnd = random.Random(28)
    P, R, B = 4, 8, 6
    m = RoutingModel(P, R, B, 64, 64)
    for r in range(B):
        m.open_request(r, rnd.randrange(0, 30))
    history = [list(map(tuple, m.route))]
    for step in range(200):
        if rnd.random() < 0.2:
            m.redirect_tails([rnd.random() < 0.4 for _ in range(P)])
        if rnd.random() < 0.1:
            act = [rnd.random() < 0.7 for _ in range(P)]
            m.set_active(act if any(act) else [1] * P)
        m.token_boundary()
        for r in range(B):
            b = m.begin[r]
            assert b[0] == 0 and all(0 < b[j + 1] - b[j] <= R for j in range(len(b) - 1))     # ranges tile [0, len]
            assert 0 <= m.len[r] - b[-1] < R                                                   # the tail has room
            assert m.append_position(r)[2] == m.len[r] - b[-1]
            assert sum(m.range_tokens_held(r, j) for j in range(len(b))) == m.len[r]
            old = history[-1][r]
            assert tuple(m.route[r][:len(old)]) == tuple(old)                                  # entries never change
        history.append([tuple(x) for x in m.route])
        m.step_commit()
    assert sum(m.partition_state()["tokens"]) == sum(m.len)
    used = [(p, s) for r in range(B) for (p, s) in m.route[r]]
    assert len(used) == len(set(used)) == m.rr_cursor


def test_no_redirect_means_begin_is_j_times_r():
    m = RoutingModel(3, 4, 2, 16, 16)
    m.open_request(0, 9)
    m.open_request(1, 0)
    for _ in range(20):
        m.token_boundary()
        m.step_commit()
    for r in range(2):
        assert m.begin[r] == [4 * j for j in range(len(m.route[r]))]
