"""Integer model of the routing table / slot allocator / append positions -- TEST INFRASTRUCTURE.

Follows PAPER.md:159-161 (routing table maps a request's token ranges to attention-node endpoints,
historical owners + live tail), :149 and :240 (route updates are published only at token boundaries;
existing ranges stay in place; future appends go to the new node), :173 (Fig. 5: [0,T/2)->A0,
[T/2,T)->A1, then [T,..)->A2 appended with nothing else changing), :145 (tail appends K/V_new before
attending).  Where the paper is silent the readings of DESIGN.md apply:

  reading 7: fixed R tokens per range, range j = [jR, (j+1)R)
  reading 8: at the boundary BEFORE appending, a request with len % R == 0 opens range len / R
  reading 9: one global round-robin cursor: the k-th range ever allocated goes to partition k % P;
             allocation order = ranges ascending within a request; requests ascending at a boundary;
             with an ACTIVE SET of partitions (the published routes of PAPER.md:216-219; "future appends use
             the new A node, while existing KV ranges remain in place", :240) the next range goes to the
             first active partition after the one used last, cyclically -- which is k % P when all are active;
             slot = per-partition LIFO free list if non-empty, else bump allocator free_head[p]++
  reading 10: exhaustion (no free slot, or range index >= max_ranges) -> error ENOSPC
  reading 24: a FULL partition is passed over by the round-robin (ENOSPC only when no active partition has a free
             slot); a request whose boundary failed has no route for its tail position: it appends nothing, is NOT
             advanced by the step commit, and every later boundary re-tries the allocation at the same position --
             the paper's "existing KV ranges remain in place ... future appends use the new A node" (:240) then
             holds again as soon as a slot is freed or a node is activated

  reading 28: "publish the route and redirect active tails on i to prewarm[i]" (Algorithm 1 l.16-17, PAPER.md:216-219;
             "at the next token boundary ... future appends use the new A node, while existing KV ranges remain in
             place", :240), taken literally: redirect_tails(parts) marks partitions; at the NEXT token boundary every
             active request whose tail range lives on a marked partition (and holds at least one token) CLOSES that
             range at its current length and continues in a new range -- beginning at position len -- on the next
             active partition.  So a range is [begin_j, begin_{j+1}) with begin_{j+1} - begin_j <= R; without
             redirects begin_j = j*R and everything above is unchanged.  A redirect that finds no free slot (or no
             free route entry) is simply not carried out: the tail stays where it is, no error.  The marks are
             consumed by that one boundary.

Pure Python, no numpy: written to be checked against the text by eye.
"""
from __future__ import annotations

from typing import Dict, List, Optional, Tuple


class RoutingError(Exception):
    pass


class RoutingModel:
    def __init__(self, n_partitions: int, range_tokens: int, max_requests: int,
                 max_ranges_per_request: int, slots_per_partition: int):
        self.P = n_partitions
        self.R = range_tokens
        self.B = max_requests
        self.Jmax = max_ranges_per_request
        self.slots = slots_per_partition
        self.len: List[int] = [-1] * max_requests          # -1 = request closed
        self.route: List[List[Tuple[int, int]]] = [[] for _ in range(max_requests)]
        self.begin: List[List[int]] = [[] for _ in range(max_requests)]    # first token position of every range
        self.redirect = set()                               # partitions whose tails move at the next boundary
        self.rr_cursor = 0                                  # ranges allocated so far
        self.rr_last = -1                                   # partition of the last allocation
        self.active = [True] * n_partitions                 # partitions that receive new ranges
        self.req_active = [True] * max_requests             # requests that take part in decode steps ("r active")
        self.free_head = [0] * n_partitions                 # bump allocator
        self.free_list: List[List[int]] = [[] for _ in range(n_partitions)]  # LIFO of released slots

    # -- allocation -----------------------------------------------------------------------------
    def _alloc(self, req: int, begin: int) -> Tuple[int, int]:
        if len(self.route[req]) >= self.Jmax:
            raise RoutingError("ENOSPC: max_ranges_per_request")
        p = None
        for i in range(1, self.P + 1):       # first active partition WITH A FREE SLOT after the last one used
            c = (self.rr_last + i) % self.P
            if self.active[c] and (self.free_list[c] or self.free_head[c] < self.slots):
                p = c
                break
        if p is None:
            raise RoutingError("ENOSPC: no active partition with a free slot")
        slot = self.free_list[p][-1] if self.free_list[p] else self.free_head[p]
        # commit
        self.rr_cursor += 1
        self.rr_last = p
        if self.free_list[p]:
            self.free_list[p].pop()
        else:
            self.free_head[p] += 1
        self.route[req].append((p, slot))
        self.begin[req].append(begin)
        return p, slot

    # -- API mirror -----------------------------------------------------------------------------
    def open_request(self, req: int, n_tokens: int) -> None:
        """Post-prefill initialisation: ceil(n/R) ranges, round-robin."""
        if self.len[req] >= 0:
            raise RoutingError("ESTATE: request already open")
        if n_tokens < 0:
            raise RoutingError("EINVAL")
        self.len[req] = n_tokens
        for j in range(-(-n_tokens // self.R)):
            self._alloc(req, j * self.R)

    def token_boundary(self) -> List[Tuple[int, int, int, int]]:
        """Open a new range for every open request whose tail position has no route: its tail range is full
        (reading 8: len % R == 0), or an earlier boundary found no slot for it (reading 24).
        Returns the events [(req, range_index, partition, slot)].  Every such request is tried, in ascending order;
        if any of them found no slot, RoutingError(ENOSPC) is raised AFTER the loop (the device latches an error word
        and carries on) and ``last_events`` holds the events of the requests that did get a range."""
        events, failed = [], None
        for r in range(self.B):
            if self.len[r] < 0 or not self.req_active[r]:
                continue
            n = self.len[r]
            if not self.route[r] or n - self.begin[r][-1] >= self.R:     # no route for position n
                try:
                    p, s = self._alloc(r, n)
                except RoutingError as e:
                    failed = failed or e
                    continue
                events.append((r, len(self.route[r]) - 1, p, s))
            elif self.route[r][-1][0] in self.redirect and n > self.begin[r][-1]:
                # reading 28: the tail range is closed at its current length; the new one starts at position n
                try:
                    p, s = self._alloc(r, n)
                except RoutingError:
                    continue                                             # not carried out: the tail stays
                events.append((r, len(self.route[r]) - 1, p, s))
        self.redirect = set()
        self.last_events = events
        if failed is not None:
            raise failed
        return events

    def append_position(self, req: int) -> Tuple[int, int, int]:
        """(partition, slot, token offset inside the range) where this step's K/V_new is written."""
        n = self.len[req]
        if n < 0:
            raise RoutingError("ESTATE: closed request")
        if not self.route[req] or n - self.begin[req][-1] >= self.R:
            raise RoutingError("ESTATE: no route for the tail position (token_boundary not called)")
        p, s = self.route[req][-1]
        return p, s, n - self.begin[req][-1]

    def step_commit(self) -> None:
        """len += 1 for every open, active request whose tail position had a route in this step (reading 24: a
        request that is waiting for a slot appended nothing and stays where it is)."""
        for r in range(self.B):
            if (self.len[r] >= 0 and self.req_active[r] and self.route[r]
                    and self.len[r] - self.begin[r][-1] < self.R):
                self.len[r] += 1

    def close_request(self, req: int) -> None:
        if self.len[req] < 0:
            raise RoutingError("ESTATE: request not open")
        for (p, s) in self.route[req]:       # ascending j
            self.free_list[p].append(s)
        self.route[req] = []
        self.begin[req] = []
        self.len[req] = -1

    def set_active(self, active) -> None:
        """Publish a new active set (scale event): future ranges only; existing routes never change."""
        if len(active) != self.P or not any(active):
            raise RoutingError("EINVAL")
        self.active = [bool(a) for a in active]

    def redirect_tails(self, parts) -> None:
        """Mark partitions (reading 28): their tails move to a new range at the next token boundary."""
        if len(parts) != self.P:
            raise RoutingError("EINVAL")
        self.redirect = {p for p in range(self.P) if parts[p]}

    def range_tokens_held(self, req: int, j: int) -> int:
        """Committed tokens of range j of an open request."""
        b = self.begin[req]
        end = b[j + 1] if j + 1 < len(b) else min(self.len[req], b[j] + self.R)
        return max(0, end - b[j])

    def set_active_requests(self, active=None) -> None:
        """Requests that take part in the following decode steps; a paused request keeps its routes and tokens."""
        self.req_active = [True] * self.B if active is None else [bool(a) for a in active]

    def partition_state(self) -> Dict[str, object]:
        """What the scaling policy monitors (Algorithm 1, l.6-9): committed tokens per partition, tails per partition."""
        tokens, tails = [0] * self.P, [0] * self.P
        for r in range(self.B):
            if self.len[r] < 0:
                continue
            for j, (p, _) in enumerate(self.route[r]):
                tokens[p] += self.range_tokens_held(r, j)
                if j == len(self.route[r]) - 1 and self.req_active[r]:   # "r active" (Algorithm 1, l.7)
                    tails[p] += 1
        return {"active": [1 if a else 0 for a in self.active], "tokens": tokens, "tails": tails}

    # -- inspection -----------------------------------------------------------------------------
    def n_ranges(self, req: int) -> int:
        return len(self.route[req])

    def locate(self, req: int, pos: int) -> Tuple[int, int, int]:
        """(partition, slot, offset) of logical token ``pos`` of a request."""
        j = max(i for i, b in enumerate(self.begin[req]) if b <= pos)
        p, s = self.route[req][j]
        return p, s, pos - self.begin[req][j]

    def snapshot(self) -> Dict[str, object]:
        part = [[-1] * self.Jmax for _ in range(self.B)]
        slot = [[-1] * self.Jmax for _ in range(self.B)]
        begin = [[-1] * self.Jmax for _ in range(self.B)]
        for r in range(self.B):
            for j, (p, s) in enumerate(self.route[r]):
                part[r][j], slot[r][j], begin[r][j] = p, s, self.begin[r][j]
        return {"len": list(self.len), "n_ranges": [len(x) for x in self.route], "part": part,
                "slot": slot, "begin": begin, "free_head": list(self.free_head), "rr_cursor": self.rr_cursor}
