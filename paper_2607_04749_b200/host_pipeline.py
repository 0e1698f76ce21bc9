"""Host-resident migration and chunked (bounded-memory) migration on top of the C ABI: stream / event plumbing only.

Both run the path as rounds of a kind-major plan (include/etc.h etc_plan_set_rounds; "state chunking ...
with on-demand buffer allocation, and eager release of source-side state"; :378 "one optimizer component at a time"):

* `HostMigration`   old shards in pinned host memory -> H2D -> whole path -> D2H -> new shards in pinned host memory.
                    Kinds are pipelined over three streams, so the upload of kind k+1, the migration of kind k and the
                    download of kind k-1 overlap (PCIe is full duplex; the copy kernels need a few % of HBM time).
                    With `needed_only=True` the plan is made first and only the source regions its slices read cross
                    PCIe (etc_upload_sources: PAPER.md:193-197, only the workload named by the instructions moves).
                    With `zero_copy=True` there are no device-side shard buffers and no DMA copies at all: the pinned
                    host buffers are handed to etc_migrate_round as they are (pinned memory is device-addressable), so
                    the copy kernels themselves read the old shards over PCIe — only the bytes their chunks name — and
                    write the new shards back over PCIe; slices that stay on their device go host -> shared memory ->
                    host in one hop, using both PCIe directions at once.
* `migrate_chunked` device-resident: for each kind, allocate its new buffers, run its rounds through one bounded
                    staging buffer, release its old buffers.  Returns the peak of live bytes, the quantity Fig. 12 of
                    the paper plots.

Every byte is moved by libetc.so's kernels or by cudaMemcpyAsync between host and device; nothing is computed here.
"""
from __future__ import annotations

from . import binding as B


def kind_order(kinds, elem_bytes):
    """Largest element size first, smallest last: the download of the last kind is the pipeline's tail."""
    return sorted(kinds, key=lambda k: (-elem_bytes[k], k))


class HostMigration:
    """Reusable pipeline for one (model, old cfg, new cfg).  `h_src` / `h_dst`: {(dev, kind): pinned uint8 host tensor}.

    run() enqueues one whole pass — (a1) layouts, (a2) cost matrix, (a3) sketch, (a4) kind-major plan + rounds, then per
    kind H2D -> (a5, a6) rounds -> D2H — and returns the plan; call torch.cuda.synchronize() (or wait on `done`)
    before reading h_dst."""

    def __init__(self, model: dict, old_cfg: dict, new_cfg: dict, h_src: dict, h_dst: dict, device=None,
                 max_staging_bytes: int = 1 << 30, flags: int = B.ETC_LOCAL_DIRECT, device_map=None,
                 d_src: dict | None = None, d_dst: dict | None = None, needed_only: bool = False, zero_copy: bool = False):
        import torch
        self.torch = torch
        self.model, self.old_cfg, self.new_cfg = model, old_cfg, new_cfg
        self.device = device or torch.device("cuda", torch.cuda.current_device())
        self.h_src, self.h_dst = h_src, h_dst
        self.flags = flags | B.ETC_KIND_MAJOR
        if zero_copy and not (flags & B.ETC_ALL_STAGED):
            self.flags |= B.ETC_ALL_DIRECT                         # one address space: a staging hop stands for nothing
        self.cap = int(max_staging_bytes)
        self.device_map = device_map
        self.needed_only = needed_only
        self.zero_copy = zero_copy
        lo, ln = B.etc_layout_create(model, old_cfg), B.etc_layout_create(model, new_cfg)
        if zero_copy:
            self.d_src = self.d_dst = {}                           # no device-side shard buffers
        else:
            self.d_src = d_src if d_src is not None else B.alloc_buffers(lo, self.device)
            self.d_dst = d_dst if d_dst is not None else B.alloc_buffers(ln, self.device)
        self.n_old, self.n_new = lo.n_dev, ln.n_dev
        self.kinds = lo.kinds()
        eb = {k: (model["param_bytes"] if k == 0 else 4) for k in self.kinds}
        self.order = kind_order(self.kinds, eb)
        self.staging = torch.empty(self.cap, dtype=torch.uint8, device=self.device)
        self.s_h2d, self.s_run, self.s_d2h = (torch.cuda.Stream(self.device) for _ in range(3))
        # planning has its own stream: etc_plan_create synchronises the stream it runs on (sizes come back to the host),
        # and on s_run that would block the host until the previous pass's rounds are done
        self.s_plan = torch.cuda.Stream(self.device)
        self.ev_plan = torch.cuda.Event()
        mk = lambda: {k: torch.cuda.Event() for k in self.kinds}
        self.ev_up, self.ev_run, self.ev_down = mk(), mk(), mk()
        self.begin, self.done = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        self.first = True
        self.h2d_bytes = sum(t.numel() for t in h_src.values())
        self.d2h_bytes = sum(t.numel() for t in h_dst.values())
        self.src_tab = B._ptr_table(self.d_src, self.n_old)
        self.dst_tab = B._ptr_table(self.d_dst, self.n_new)
        self.h_src_tab = B._ptr_table(self.h_src, self.n_old)
        self.h_dst_tab = B._ptr_table(self.h_dst, self.n_new)

    def _plan(self):
        """(a1)-(a4) on the planning stream; s_run is made to wait for it."""
        with self.torch.cuda.stream(self.s_plan):
            lo, ln = B.etc_layout_create(self.model, self.old_cfg), B.etc_layout_create(self.model, self.new_cfg)
            if self.device_map is None:
                ov, _, _ = B.etc_cost_matrix(lo, ln, stream=self.s_plan)
                dm, _ = B.etc_sketch(ov, stream=self.s_plan)
            else:
                dm = self.device_map
            plan = B.etc_plan_create(lo, ln, dm, self.flags, stream=self.s_plan)
            rounds = B.etc_plan_set_rounds(plan, self.cap, stream=self.s_plan)
            self.ev_plan.record(self.s_plan)
        self.s_run.wait_event(self.ev_plan)
        return plan, rounds

    def run(self):
        if self.zero_copy:
            return self._run_zero_copy()
        if self.needed_only:
            return self._run_needed_only()
        torch = self.torch
        # uploads: kind by kind; a buffer may be overwritten only after the previous pass's rounds have read it
        with torch.cuda.stream(self.s_h2d):
            if self.first:
                self.begin.record(self.s_h2d)
            for k in self.order:
                if not self.first:
                    self.s_h2d.wait_event(self.ev_run[k])
                for (d, kk), t in self.d_src.items():
                    if kk == k:
                        t.copy_(self.h_src[(d, kk)], non_blocking=True)
                self.ev_up[k].record(self.s_h2d)
        # planning (metadata only) overlaps the first upload
        plan, rounds = self._plan()
        with torch.cuda.stream(self.s_run):
            for k in self.order:
                self.s_run.wait_event(self.ev_up[k])
                if not self.first:
                    self.s_run.wait_event(self.ev_down[k])         # previous pass's download of these buffers
                for i, r in enumerate(rounds):
                    if r.kind == k:
                        B.etc_migrate_round(plan, i, self.src_tab, self.dst_tab, self.staging, stream=self.s_run)
                self.ev_run[k].record(self.s_run)
        with torch.cuda.stream(self.s_d2h):
            for k in self.order:
                self.s_d2h.wait_event(self.ev_run[k])
                for (n, kk), t in self.d_dst.items():
                    if kk == k:
                        self.h_dst[(n, kk)].copy_(t, non_blocking=True)
                self.ev_down[k].record(self.s_d2h)
            self.done.record(self.s_d2h)
        self.first = False
        self.plan = plan
        return plan


    def _run_zero_copy(self):
        """Plan, then the rounds with the pinned HOST buffers as source and destination tables: every byte is moved by
        the copy kernels, over PCIe; the device holds only the plan's tables and the bounded staging buffer."""
        if self.first:
            self.begin.record(self.s_plan)
        plan, rounds = self._plan()
        for i in range(len(rounds)):
            B.etc_migrate_round(plan, i, self.h_src_tab, self.h_dst_tab, self.staging, stream=self.s_run)
        self.done.record(self.s_run)
        st = plan.stats
        self.h2d_bytes = st.local_bytes + st.remote_bytes          # payload bytes the kernels read from host memory
        self.d2h_bytes = st.local_bytes + st.remote_bytes + st.fill_bytes
        self.first = False
        self.plan = plan
        return plan

    def _run_needed_only(self):
        """Plan first (metadata, < 1 ms), then per kind: upload the regions the plan reads -> rounds -> download.
        The three queues are fed kind by kind: a stream accepts only so many pending copies before the enqueueing call
        blocks, and an upload is thousands of region copies, so the rounds and the download of kind k must be queued
        before the upload of kind k+1 is."""
        torch = self.torch
        if self.first:
            self.begin.record(self.s_plan)
        plan, rounds = self._plan()
        self.h2d_bytes = 0
        for k in self.order:
            if not self.first:
                self.s_h2d.wait_event(self.ev_run[k])              # the previous pass's rounds have read these buffers
            self.h2d_bytes += B.etc_upload_sources(plan, self.h_src_tab, self.src_tab, k, stream=self.s_h2d)
            self.ev_up[k].record(self.s_h2d)
            self.s_run.wait_event(self.ev_up[k])
            if not self.first:
                self.s_run.wait_event(self.ev_down[k])             # the previous pass's download of these buffers
            for i, r in enumerate(rounds):
                if r.kind == k:
                    B.etc_migrate_round(plan, i, self.src_tab, self.dst_tab, self.staging, stream=self.s_run)
            self.ev_run[k].record(self.s_run)
            self.s_d2h.wait_event(self.ev_run[k])
            with torch.cuda.stream(self.s_d2h):
                for (n, kk), t in self.d_dst.items():
                    if kk == k:
                        self.h_dst[(n, kk)].copy_(t, non_blocking=True)
            self.ev_down[k].record(self.s_d2h)
        self.done.record(self.s_d2h)
        self.first = False
        self.plan = plan
        return plan


def migrate_chunked(plan, new_layout, src_bufs: dict, max_staging_bytes: int, device=None, stream=None, fill=None):
    """Device-resident chunked migration with eager release.  `src_bufs` is CONSUMED: the buffers of a kind are dropped
    from the dict as soon as the kind's last round has been enqueued (torch's caching allocator frees them in stream
    order).  Returns (dst_bufs, info) with info = {"rounds", "peak_live_bytes", "staging_bytes", "old_bytes",
    "new_bytes"}; peak_live_bytes counts old + new + staging bytes alive at the worst moment."""
    import torch
    device = device or torch.device("cuda", torch.cuda.current_device())
    rounds = B.etc_plan_set_rounds(plan, max_staging_bytes, stream=stream)
    stg_bytes = max((r.staging_bytes for r in rounds), default=0)
    staging = torch.empty(max(stg_bytes, 16), dtype=torch.uint8, device=device)
    old_bytes = sum(t.numel() for t in src_bufs.values())
    live = old_bytes + stg_bytes
    peak = live
    dst = {}
    new_total = 0
    for k in sorted({r.kind for r in rounds} | {key[1] for key in src_bufs}):
        mine = {}
        for n in range(new_layout.n_dev):                          # on-demand allocation of the kind's new buffers
            nb = new_layout.buffer_bytes(n, k)
            if nb > 0:
                mine[(n, k)] = torch.empty(nb, dtype=torch.uint8, device=device) if fill is None else \
                    torch.full((nb,), fill, dtype=torch.uint8, device=device)
                live += nb; new_total += nb
        peak = max(peak, live)
        dst.update(mine)
        for i, r in enumerate(rounds):
            if r.kind == k:
                B.etc_migrate_round(plan, i, src_bufs, dst, staging, stream=stream)
        for key in [key for key in src_bufs if key[1] == k]:       # eager release of the source side
            live -= src_bufs[key].numel()
            del src_bufs[key]
    return dst, {"rounds": len(rounds), "peak_live_bytes": peak, "staging_bytes": stg_bytes, "old_bytes": old_bytes,
                 "new_bytes": new_total}
