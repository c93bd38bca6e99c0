"""DecodeLoop — drives one D-instance through the decode steps of a BASELINE.json workload.

Scheduling and argument marshalling only: every byte of KV is moved, and every attention
output computed, by the kernels behind the C-ABI (``binding``).  ``bench.py`` times this loop
and the ``-m gpu`` full-size parity tests run the same loop, so the launch configuration that
is measured is the one that is checked.

One step (SURVEY §8(a), rows a1-a6; PAPER.md:200, :219-223 producer/consumer balance):
    host      retire `ingest_per_step` finished requests           kv_free        (a6)
    stream B  ingest `ingest_per_step` prefill-completed requests  kv_ingest      (a1, a2)
              (they join the decode batch at the NEXT step, so the copy overlaps attention)
    stream A  reserve the step's token for every request and, for each layer, append + attention over len+1:
              ONE host call, paged_decode_step_layers(KV_STEP_RESERVE) — a1 on the host, then one launch per
              layer (a3, a4, a5 fused), issued back to back with programmatic dependent launch
              (``layered=False``: kv_reserve + one paged_decode_step call per layer;
               ``fused=False``: kv_ingest n=1 then paged_decode_attention, two or three launches per layer)
The decode batch keeps its size: the requests retired at step s are replaced by the ones
ingested during step s-1.  With ``streams=1`` everything runs on stream A in program order.

Cross-stream ordering (the hazards kv_free's contract names): stream B waits for the end of
step s-1 on A before it writes blocks recycled from requests retired at step s; stream A waits
for B's ingest of step s-1 before it attends over the requests that joined.

Contents are functions of logical position (``workloads``): request `uid`'s token t is
kv_values(seed, kind, content_uid[uid], ...), so a checker can regenerate any request on the
CPU.  Newly arriving requests draw their content from a pre-generated bank of
``bank_steps * ingest_per_step`` sources that is cycled (the bank entry fixes both the length
and the content uid); this bounds device memory without putting a generator in the timed region.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np
import torch

from . import binding as B
from . import workloads as W

BANK_UID0 = 1 << 24  # content uids of bank entries (initial requests use their own id)


def _align(x: int, a: int = 256) -> int:
    return (x + a - 1) // a * a


@dataclass
class StepPlan:
    """Everything step s needs on the host, precomputed from the seeded schedule."""
    retire: np.ndarray        # int64 ids freed at the start of the step
    arrive: np.ndarray        # int64 ids ingested during the step (join the batch next step)
    arrive_bank: np.ndarray   # bank entry of each arrival
    batch: np.ndarray         # int64 ids attended in this step (fixed size)
    lens_after: np.ndarray    # int64 context length of each batch row AFTER this step's append
    attn_bytes_layer: int     # algorithmic bytes of one layer's attention
    append_bytes: int         # 2 x source bytes of the appends, all layers
    ingest_bytes: int         # 2 x source bytes of the arrivals, all layers
    ingest_tokens: int


@dataclass
class Schedule:
    n0: np.ndarray
    bank_lens: np.ndarray
    prime: StepPlan | None
    steps: list = field(default_factory=list)
    content_uid: dict = field(default_factory=dict)
    peak_blocks: int = 0


kv_token_bytes_layer = W.kv_token_bytes_layer
attention_bytes = W.attention_bytes


def build_schedule(w: W.Workload, n_steps: int, bank_steps: int, salt: int = 0, host_from: int | None = None,
                   host_bank_steps: int = 2, fp8: bool = False) -> Schedule:
    """Seeded, host-only simulation of which requests retire / arrive / decode at every step.
    Steps >= host_from (the host-buffer steps) cycle over the first `host_bank_steps` bank steps only,
    which are the ones mirrored in pinned host memory."""
    host_from = n_steps if host_from is None else host_from
    rng = w.rng(1000 + salt)
    n0 = w.draw_lengths(salt=salt)
    k = w.ingest_per_step
    bank_lens = w.draw_lengths(n=max(1, bank_steps * k), salt=500 + salt) if k else np.zeros(0, np.int64)
    sch = Schedule(n0=n0, bank_lens=bank_lens, prime=None)
    lens = {i: int(n) for i, n in enumerate(n0)}
    for i in lens:
        sch.content_uid[i] = i
    order = list(range(w.batch))          # FIFO arrival order of the decode batch
    next_id = w.batch
    # per token: K+V bf16 source bytes read + pool bytes written (all layers)
    row = 2 * w.num_layers * w.num_kv_heads * w.head_dim * 2 + w.num_layers * kv_token_bytes_layer(w, fp8)
    blocks = lambda n: (n + w.block_size - 1) // w.block_size
    live_blocks = sum(blocks(n) for n in lens.values())
    sch.peak_blocks = live_blocks
    pending: list[int] = []

    def arrivals(step_idx: int):
        nonlocal next_id, live_blocks
        ids, banks = [], []
        for j in range(k):
            cyc = min(host_bank_steps, bank_steps) if step_idx >= host_from else bank_steps
            e = (step_idx % cyc) * k + j
            ids.append(next_id)
            banks.append(e)
            lens[next_id] = int(bank_lens[e])
            sch.content_uid[next_id] = BANK_UID0 + e
            live_blocks += blocks(lens[next_id])
            next_id += 1
        return ids, banks

    if k:  # priming: the arrivals that join at step 0 (ingested before the timed region)
        ids, banks = arrivals(-1)
        pending = ids
        sch.prime = StepPlan(np.zeros(0, np.int64), np.asarray(ids, np.int64), np.asarray(banks, np.int64),
                             np.zeros(0, np.int64), np.zeros(0, np.int64), 0, 0,
                             sum(lens[i] for i in ids) * row, sum(lens[i] for i in ids))
        sch.peak_blocks = max(sch.peak_blocks, live_blocks)
    for s in range(n_steps):
        retire: list[int] = []
        if k:
            if w.pool_hbm_frac > 0:   # config 5: finished requests are sampled uniformly
                pick = sorted(rng.choice(len(order), size=k, replace=False).tolist(), reverse=True)
                retire = [order.pop(i) for i in pick]
            else:                     # config 3: the oldest finish first
                retire, order = order[:k], order[k:]
            for i in retire:
                live_blocks -= blocks(lens.pop(i))
            order += pending
            ids, banks = arrivals(s)
            pending = ids
        else:
            ids, banks = [], []
        batch = np.asarray(order, np.int64)
        for i in order:               # a3: one appended token per request, then attend over len+1 (A3)
            live_blocks += blocks(lens[i] + 1) - blocks(lens[i])
            lens[i] += 1
        la = np.asarray([lens[i] for i in order], np.int64)
        sch.peak_blocks = max(sch.peak_blocks, live_blocks)
        sch.steps.append(StepPlan(np.asarray(retire, np.int64), np.asarray(ids, np.int64),
                                  np.asarray(banks, np.int64), batch, la, attention_bytes(w, la, fp8),
                                  len(order) * row, sum(lens[i] for i in ids) * row,
                                  sum(lens[i] for i in ids)))
    return sch


class DecodeLoop:
    """A pool, its resident decode batch and the pre-generated inputs of `n_steps` decode steps."""

    HOST_BANK_STEPS = 2

    def __init__(self, w: W.Workload, n_steps: int, n_host_steps: int = 0, device="cuda:0", streams: int = 2,
                 salt: int = 0, bank_bytes: int = 24 << 30, profile: bool = True, options: dict | None = None,
                 sentinel: int | None = None, fused: bool = True, kv_dtype: int = B.KV_DTYPE_BF16, layered: bool = True,
                 inline_ingest: bool = False):
        """Steps [0, n_steps) take their inputs from device memory; steps [n_steps, n_steps + n_host_steps)
        take them from pinned host memory through the *_host entry points."""
        self.fp8 = kv_dtype == B.KV_DTYPE_FP8_E4M3
        self.w, self.dev, self.salt, self.fused = w, torch.device(device), salt, fused
        self.layered = layered and fused
        self.host_from, self.n_steps = n_steps, n_steps + n_host_steps
        self.two_streams = streams >= 2 and w.ingest_per_step > 0
        # device-resident arrivals ingested in line on the decode stream (host-resident ones stay on stream B: their copy
        # is PCIe-bound and overlaps for free).  Worth it on FP8 pools, see bench.py --streams
        self.inline_ingest = inline_ingest and self.two_streams
        L, Hkv, Hq, d, k = w.num_layers, w.num_kv_heads, w.num_q_heads, w.head_dim, w.ingest_per_step
        self.tok_bytes = L * Hkv * d * 2                      # one tensor (K or V), one token, all layers
        mean_len = float(np.mean(w.draw_lengths(n=4096, salt=900)))
        per_step = max(1.0, 2 * self.tok_bytes * mean_len * max(k, 1))
        self.bank_steps = int(min(8, max(2, bank_bytes // per_step))) if k else 0
        self.sched = build_schedule(w, self.n_steps, max(self.bank_steps, 1), salt, self.host_from,
                                    self.HOST_BANK_STEPS, self.fp8)

        # ---- pool ----
        block_bytes = L * w.block_size * kv_token_bytes_layer(w, self.fp8)
        if w.pool_hbm_frac > 0:
            total = torch.cuda.get_device_properties(self.dev).total_memory
            num_blocks = int(total * w.pool_hbm_frac) // block_bytes
            assert num_blocks >= self.sched.peak_blocks, "workload does not fit the pool"
        else:
            num_blocks = max(int(self.sched.peak_blocks * w.pool_slack), self.sched.peak_blocks + 64)
        self.cfg = B.PoolConfig(num_layers=L, num_q_heads=Hq, num_kv_heads=Hkv, head_dim=d, num_blocks=num_blocks,
                                max_requests=w.batch + 3 * k + 32,
                                max_blocks_per_request=(w.max_len + self.n_steps + w.block_size) // w.block_size + 1,
                                alloc_seed=w.seed + salt, kv_dtype=kv_dtype)
        self.pool = B.KVPool(self.cfg, device=self.dev)
        if sentinel is not None:
            self.pool.slab[: self.pool.kv_bytes].view(torch.int16).fill_(sentinel)
        for key, val in (options or {}).items():
            self.pool.set_option(key, val)
        if profile:
            self.pool.set_option("profile", 1)
        # decode (A) outranks bulk ingest (B): the block scheduler hands B's CTAs the SM time A leaves idle
        self.sA = torch.cuda.Stream(self.dev, priority=-1)
        self.sB = torch.cuda.Stream(self.dev, priority=0) if self.two_streams else self.sA
        self.evA = [torch.cuda.Event() for _ in range(4)]      # end of step on A (ring)
        self.evB = [torch.cuda.Event() for _ in range(4)]      # end of ingest on B (ring)
        self.step_idx = 0
        self._fill_initial()
        self._make_bank()
        self._make_step_inputs()
        if self.sched.prime is not None:                        # arrivals that join at step 0
            self._ingest_arrivals(self.sched.prime, self.sB)
        torch.cuda.synchronize(self.dev)
        self.pool.profile_reset()

    # ---- setup ------------------------------------------------------------------------------
    def _src(self, uid: int, t0: int, t1: int, device=None):
        w = self.w
        dev = self.dev if device is None else device
        return (W.kv_values(w.seed, W.KIND_K, uid, w.num_kv_heads, w.head_dim, 0, w.num_layers, t0, t1, dev),
                W.kv_values(w.seed, W.KIND_V, uid, w.num_kv_heads, w.head_dim, 0, w.num_layers, t0, t1, dev))

    def _fill_initial(self):
        """Resident batch before step 0, through kv_ingest.  `fragmented` (config 4): requests grow
        round-robin in 64-token slices on the permuted free list, so consecutive logical blocks of
        a request are never neighbours in memory."""
        w, n0 = self.w, self.sched.n0
        with torch.cuda.stream(self.sA):
            if not w.fragmented:
                group, gbytes = [], 0
                for i, n in enumerate(n0):
                    k_, v_ = self._src(i, 0, int(n))
                    group.append((i, k_, v_))
                    gbytes += 2 * k_.numel() * 2
                    if gbytes > (4 << 30) or i == len(n0) - 1:
                        self.pool.ingest([g[0] for g in group], [g[1] for g in group], [g[2] for g in group],
                                         stream=self.sA)
                        self.sA.synchronize()
                        group, gbytes = [], 0
                return
            sl = 64
            L, Hkv, d = w.num_layers, w.num_kv_heads, w.head_dim
            slices = []                                           # per request: [n_full][L][Hkv][sl][d] + tail
            for i, n in enumerate(n0):
                n = int(n)
                k_, v_ = self._src(i, 0, n)
                nf = n // sl
                cut = lambda x: x[:, :, : nf * sl].reshape(L, Hkv, nf, sl, d).permute(2, 0, 1, 3, 4).contiguous()
                tail = lambda x: x[:, :, nf * sl:].contiguous()
                slices.append((n, nf, cut(k_), cut(v_), tail(k_), tail(v_)))
            rounds = max((int(n) + sl - 1) // sl for n in n0)
            sbytes = L * Hkv * sl * d * 2
            for r in range(rounds):
                ids, nt, kp, vp = [], [], [], []
                for i, (n, nf, kc, vc, kt, vt) in enumerate(slices):
                    if r < nf:
                        ids.append(i); nt.append(sl); kp.append(kc.data_ptr() + r * sbytes); vp.append(vc.data_ptr() + r * sbytes)
                    elif r == nf and n > nf * sl:
                        ids.append(i); nt.append(n - nf * sl); kp.append(kt.data_ptr()); vp.append(vt.data_ptr())
                if ids:
                    B.kv_ingest(self.pool.handle, ids, nt, kp, vp, 0, L, self.sA.cuda_stream)
            self.sA.synchronize()

    def _make_bank(self):
        """Sources of the arriving requests: bank entry e = (length bank_lens[e], content uid BANK_UID0+e)."""
        self.bank = []
        self.bank_host = []
        for e, n in enumerate(self.sched.bank_lens if self.w.ingest_per_step else []):
            with torch.cuda.stream(self.sA):
                k_, v_ = self._src(BANK_UID0 + e, 0, int(n))
            self.sA.synchronize()
            self.bank.append((k_, v_))
            if self.n_steps > self.host_from and e < self.HOST_BANK_STEPS * self.w.ingest_per_step:
                kh = torch.empty(k_.shape, dtype=k_.dtype, pin_memory=True).copy_(k_)
                vh = torch.empty(v_.shape, dtype=v_.dtype, pin_memory=True).copy_(v_)
                self.bank_host.append((kh, vh))
        if self.bank_host:
            k = self.w.ingest_per_step
            need = max(sum(2 * _align(self.tok_bytes * int(n)) for n in self.sched.bank_lens[s * k:(s + 1) * k])
                       for s in range(min(self.HOST_BANK_STEPS, self.bank_steps)))
            self.stage_B = torch.empty(need, dtype=torch.uint8, device=self.dev)

    def _make_step_inputs(self):
        """Per step: q [L][B][Hq][d], appended-token K/V [L][B][Hkv][d] (values by logical position)."""
        w = self.w
        L, Bn, Hq, Hkv, d = w.num_layers, w.batch, w.num_q_heads, w.num_kv_heads, w.head_dim
        self.q, self.k_new, self.v_new, self.out = [], [], [], []
        with torch.cuda.stream(self.sA):
            for s, sp in enumerate(self.sched.steps):
                host = s >= self.host_from
                pin = dict(pin_memory=True) if host else dict(device=self.dev)
                cu = [self.sched.content_uid[int(i)] for i in sp.batch]
                pos = sp.lens_after - 1
                kn = W.kv_values_at(w.seed, W.KIND_K, cu, pos, Hkv, d, 0, L, self.dev)
                vn = W.kv_values_at(w.seed, W.KIND_V, cu, pos, Hkv, d, 0, L, self.dev)
                q = torch.stack([W.q_values(w.seed + self.salt, s, l, Bn, Hq, d, self.dev) for l in range(L)])
                if host:
                    kn, vn, q = (torch.empty(x.shape, dtype=x.dtype, **pin).copy_(x) for x in (kn, vn, q))
                self.k_new.append(kn); self.v_new.append(vn); self.q.append(q)
                self.out.append(torch.empty((L, Bn, Hq, d), dtype=torch.bfloat16, **pin))
        self.sA.synchronize()
        self.row_new = Hkv * d * 2
        self.q_layer_bytes = Bn * Hq * d * 2
        self._offs = np.arange(Bn, dtype=np.uint64) * np.uint64(self.row_new)
        self._ones = np.ones(Bn, dtype=np.int32)
        if self.n_steps > self.host_from:
            self.stage_A = torch.empty(2 * _align(Bn * self.row_new) + 2 * _align(self.q_layer_bytes),
                                       dtype=torch.uint8, device=self.dev)

    # ---- one step ---------------------------------------------------------------------------
    def _ingest_arrivals(self, sp: StepPlan, stream, host: bool = False):
        if sp.arrive.size == 0:
            return
        L = self.w.num_layers
        nt = self.sched.bank_lens[sp.arrive_bank].astype(np.int32)
        if host:
            kp = np.asarray([self.bank_host[e][0].data_ptr() for e in sp.arrive_bank], dtype=np.uint64)
            vp = np.asarray([self.bank_host[e][1].data_ptr() for e in sp.arrive_bank], dtype=np.uint64)
            B.kv_ingest_host(self.pool.handle, sp.arrive, nt, kp, vp, 0, L, self.stage_B.data_ptr(),
                             self.stage_B.numel(), stream.cuda_stream)
        else:
            kp = np.asarray([self.bank[e][0].data_ptr() for e in sp.arrive_bank], dtype=np.uint64)
            vp = np.asarray([self.bank[e][1].data_ptr() for e in sp.arrive_bank], dtype=np.uint64)
            B.kv_ingest(self.pool.handle, sp.arrive, nt, kp, vp, 0, L, stream.cuda_stream)

    def step(self):
        """Enqueue decode step `self.step_idx` (returns without synchronising)."""
        s = self.step_idx
        sp = self.sched.steps[s]
        host = s >= self.host_from
        h, A, Bs = self.pool.handle, self.sA, self.sB
        L = self.w.num_layers
        if sp.retire.size:
            B.kv_free(h, sp.retire)                                     # a6 (host)
        if sp.arrive.size:                                               # a1 + a2 on stream B (or in line on A)
            S = A if (self.inline_ingest and not host) else Bs
            if self.two_streams and s > 0 and S is not A:
                S.wait_event(self.evA[(s - 1) % 4])                      # recycled blocks were read by step s-1
            self._ingest_arrivals(sp, S, host)
            if self.two_streams:
                self.evB[s % 4].record(S)
        if self.two_streams and s > 0:
            A.wait_event(self.evB[(s - 1) % 4])                          # joiners of this step were ingested at s-1
        kn, vn, q, out = self.k_new[s], self.v_new[s], self.q[s], self.out[s]
        a = A.cuda_stream
        lay_kv = self.w.batch * self.row_new
        qb = self.q_layer_bytes
        if self.layered and not host:                                                              # a1 + L x (a3 + a4 + a5)
            B.paged_decode_step_layers(h, 0, L, sp.batch, q.data_ptr(), kn.data_ptr(), vn.data_ptr(), out.data_ptr(),
                                       qb, lay_kv, 0.0, B.KV_STEP_RESERVE, a)
            L = 0
        elif self.fused:
            B.kv_reserve(h, sp.batch, self._ones)                                                  # a1 (host)
        for l in range(L):
            kl, vl = kn.data_ptr() + l * lay_kv, vn.data_ptr() + l * lay_kv
            ql, ol = q.data_ptr() + l * qb, out.data_ptr() + l * qb
            if self.fused and host:
                B.paged_decode_step_host(h, l, sp.batch, ql, kl, vl, ol, 0.0, self.stage_A.data_ptr(),
                                         self.stage_A.numel(), a)                                  # a3 + a4 + a5
            elif self.fused:
                B.paged_decode_step(h, l, sp.batch, ql, kl, vl, ol, 0.0, a)                        # a3 + a4 + a5
            elif host:
                off = 2 * _align(lay_kv)
                B.kv_ingest_host(h, sp.batch, self._ones, self._offs + np.uint64(kl), self._offs + np.uint64(vl),
                                 l, 1, self.stage_A.data_ptr(), off, a)                            # a3
                B.paged_decode_attention_host(h, l, sp.batch, ql, ol, 0.0, self.stage_A.data_ptr() + off,
                                              self.stage_A.numel() - off, a)                       # a4 + a5
            else:
                B.kv_ingest(h, sp.batch, self._ones, self._offs + np.uint64(kl), self._offs + np.uint64(vl),
                            l, 1, a)                                                               # a3
                B.paged_decode_attention(h, l, sp.batch, ql, ol, 0.0, a)                           # a4 + a5
        if self.two_streams:
            self.evA[s % 4].record(A)
        self.step_idx += 1

    def join(self):
        """Make stream A wait for everything enqueued on stream B (end of a timed region)."""
        if self.two_streams:
            ev = torch.cuda.Event()
            ev.record(self.sB)
            self.sA.wait_event(ev)

    # ---- accounting -------------------------------------------------------------------------
    def bytes_of_steps(self, lo: int, hi: int) -> dict:
        sps = self.sched.steps[lo:hi]
        L = self.w.num_layers
        return dict(attn=sum(sp.attn_bytes_layer for sp in sps) * L,
                    append=sum(sp.append_bytes for sp in sps),
                    ingest=sum(sp.ingest_bytes for sp in sps),
                    tokens=sum(len(sp.batch) for sp in sps),
                    ingest_tokens=sum(sp.ingest_tokens for sp in sps))

    def io_bytes(self, lo: int, hi: int) -> tuple[int, int]:
        """(host->device, device->host) bytes of host-buffer steps [lo, hi), counted from the tensors copied:
        q, the appended K/V rows and the arriving requests' K/V in; the attention outputs back."""
        L, h2d, d2h = self.w.num_layers, 0, 0
        for s in range(lo, hi):
            sp = self.sched.steps[s]
            h2d += self.q[s].numel() * 2 + self.k_new[s].numel() * 2 + self.v_new[s].numel() * 2
            h2d += 2 * self.tok_bytes * sp.ingest_tokens
            d2h += self.out[s].numel() * 2
        return h2d, d2h

    def close(self):
        torch.cuda.synchronize(self.dev)
        self.pool.close()
