"""Target sharding of ONE event over several GPUs (include/gcoreccd.h
"Target sharding").  Host orchestration only: every step of the path runs in the library's kernels.

Per step and rank:   shard_local(msg)  ->  exchange.gather(msg) -> [G messages]  ->  shard_commit([G messages])
The state is replicated, the rows of eq. 6 are not: rank g advances the targets of its share against
all sources and contributes its survivors; the concatenation in rank order is the next state.  Images, counters and
collection records are rank-local and summed once at the end (integers, so the sum is exact).

Exchanges (how the G messages reach a rank):
  DistExchange     torch.distributed.all_gather_into_tensor on the message bytes: NCCL over NVLink on GPUs, gloo in
                   the CPU tests (tests/test_sharded_gloo.py drives it with an oracle-backed engine).
  SymmMemExchange  the messages live in torch symmetric memory; shard_commit reads the PEERS' buffers directly, so
                   the all-gather is fused into the commit kernel's loads over NVLink, and the kernel waits on the
                   message headers itself (a release-ordered word per message): no collective and no barrier is
                   left in a step.  Exercised at world size 1 only (tests, bench --exchange symm): this build's
                   boxes have one GPU, and ranks that wait on one another must not share a GPU (B200_PROFILING.md).
  VirtualRanks     G handles on ONE device stepped one after the other on one stream, messages passed by pointer:
                   the same kernels and the same pointer-table commit as the multi-GPU path, with no kernel ever
                   waiting on another (B200_PROFILING.md: emulate ranks sequentially, never concurrently).

An "engine" is anything with set_shard / shard_message_bytes / shard_local(ptr, bytes) / shard_commit(ptrs, bytes) /
state() / read_image() / read_collected(): binding.Gcoreccd on GPUs.
"""
import numpy as np

REFRESH_STEPS = 32          # steps between host reads of n_active (message size and termination follow it)
HEADER_BYTES = 256


def share_of(n_active, rank, world):
    """[t0, t0+nt): the targets rank owns at n_active (mirror of gc_common.cuh shard_range, for tests and sizing)."""
    T = (int(n_active) + 255) // 256
    a, b = (T * rank // world) * 256, (T * (rank + 1) // world) * 256
    lo, hi = min(a, n_active), min(b, n_active)
    return lo, hi - lo


class DistExchange:
    """all-gather of the message bytes through torch.distributed (backend of the initialised process group)."""

    def __init__(self, torch, device, max_bytes, world, group=None):
        import torch.distributed as dist
        self.dist, self.group, self.world = dist, group, world
        self.recv = torch.empty(world * max_bytes, dtype=torch.uint8, device=device)

    def gather(self, msg, nbytes):
        out = self.recv[: self.world * nbytes]
        self.dist.all_gather_into_tensor(out, msg[:nbytes], group=self.group)
        base = out.data_ptr()
        return [base + g * nbytes for g in range(self.world)]

    def after_commit(self):
        pass


class SymmMemExchange:
    """Peer-mapped message buffers (torch.distributed._symmetric_memory): commit loads cross NVLink directly."""

    def __init__(self, torch, device, max_bytes, world, group_name=None):
        import torch.distributed as dist
        import torch.distributed._symmetric_memory as symm
        self.world = world
        name = group_name or dist.group.WORLD.group_name
        self.buf = symm.empty(2 * max_bytes, dtype=torch.uint8, device=device)      # two messages, alternated
        self.hdl = symm.rendezvous(self.buf, name)
        self.max_bytes = max_bytes
        self.k = 0

    def message(self):
        """The local buffer the next shard_local must write (inside the symmetric allocation)."""
        off = (self.k & 1) * self.max_bytes
        return self.buf[off: off + self.max_bytes]

    flag_synchronised = True                  # ShardedEvent then switches the engine's commit kernel to header waits

    def gather(self, msg, nbytes):
        """No collective and no barrier: shard_commit reads the peers' buffers and waits on their headers by itself
        (include/gcoreccd.h gcoreccd_set_shard_wait); the host only hands it the G pointers."""
        off = (self.k & 1) * self.max_bytes
        ptrs = [int(p) + off for p in self.hdl.buffer_ptrs]
        self.k += 1
        return ptrs

    def after_commit(self):
        pass                                  # the other half is written next step; its readers finished a barrier ago


class ShardedEvent:
    """One rank's view of an event sharded over `world` ranks."""

    def __init__(self, engine, rank, world, exchange_factory, alloc):
        """alloc(nbytes) -> uint8 tensor on the engine's device; exchange_factory(max_bytes) -> exchange."""
        self.e, self.rank, self.world = engine, int(rank), int(world)
        engine.set_shard(rank, world)
        self._alloc, self._xf = alloc, exchange_factory
        self.x, self.msgs, self.max_bytes, self.k = None, None, 0, 0
        self.nbytes = 0

    def _prepare(self):
        """(Re)size the messages for the current bound on n_active; called after loads and refreshes."""
        self.nbytes = self.e.shard_message_bytes()
        if self.nbytes > self.max_bytes:
            self.max_bytes = self.nbytes
            with self._on_engine_stream():   # buffers allocated by torch belong to the stream that uses them
                if self.x is not None and getattr(self.x, "flag_synchronised", False):
                    self.e._torch.cuda.synchronize()     # a larger symmetric buffer replaces one peers may still read
                self.x = self._xf(self.max_bytes)
                if getattr(self.x, "flag_synchronised", False):
                    self.e.set_shard_wait(True)
                if not hasattr(self.x, "message"):
                    self.msgs = [self._alloc(self.max_bytes), self._alloc(self.max_bytes)]

    def load_carriers(self, xyz):
        """Every rank loads the same holes in the same order."""
        self.e.load_carriers(xyz)
        self.refresh()

    def refresh(self):
        st = self.e.state()                   # synchronises; updates the library's bound on n_active
        self._prepare()
        return st

    def _on_engine_stream(self):
        """The exchange (an NCCL all-gather, a symmetric-memory barrier) is enqueued on torch's CURRENT stream, the
        library's kernels on the handle's stream: make them the same stream for the duration of a step, so that
        shard_local -> gather -> shard_commit are ordered by the stream and nothing else."""
        st = getattr(self.e, "_stream", None)
        if st is None:                       # an engine without a CUDA stream (the CPU test engine)
            import contextlib
            return contextlib.nullcontext()
        return self.e._torch.cuda.stream(st)

    def step(self, n=1):
        if self.x is None:
            self._prepare()
        with self._on_engine_stream():
            for _ in range(int(n)):
                msg = self.x.message() if hasattr(self.x, "message") else self.msgs[self.k & 1]
                self.k += 1
                self.e.shard_local(msg.data_ptr(), self.nbytes)
                ptrs = self.x.gather(msg, self.nbytes)
                self.e.shard_commit(ptrs, self.nbytes)
                self.x.after_commit()

    def run_to_collection(self, max_steps=10 ** 9):
        st = self.refresh()
        step0, done = st["step"], 0
        while st["n_active"] > 0 and done < max_steps:
            self.step(min(REFRESH_STEPS, max_steps - done))
            st = self.refresh()
            done = st["step"] - step0
        return done, st["n_active"]

    # ---- results: integer sums over ranks
    def totals(self, reduce_sum):
        """reduce_sum(np.int64 array) -> summed over ranks.  Returns the event's global counters."""
        st = self.e.state()
        v = reduce_sum(np.array([st["n_collected"], st["n_out_of_window"], st["pair_interactions"]], dtype=np.int64))
        return {"step": st["step"], "n_active": st["n_active"], "n_loaded": st["n_loaded"], "n_collected": int(v[0]),
                "n_out_of_window": int(v[1]), "pair_interactions": int(v[2])}

    def image(self, reduce_sum):
        img, _ = self.e.read_image()
        return reduce_sum(np.asarray(img, dtype=np.int64)).astype(np.uint32)


def dist_reduce_sum(torch, device, group=None):
    import torch.distributed as dist

    def f(a):
        t = torch.from_numpy(np.ascontiguousarray(a)).to(device)
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
        return t.cpu().numpy()
    return f


class VirtualRanks:
    """G engines on one device, stepped sequentially on one stream (module docstring).  For parity tests and for
    timing the per-rank kernels of a G-way run on a single GPU."""

    def __init__(self, engines, alloc):
        self.es, self.G = list(engines), len(engines)
        if len({e._stream.cuda_stream for e in self.es}) != 1:
            # every rank's commit reads every other rank's message: stream order IS the synchronisation here
            raise ValueError("VirtualRanks: all engines must be created on the same CUDA stream")
        for g, e in enumerate(self.es):
            e.set_shard(g, self.G)
        self._alloc, self.max_bytes, self.msgs, self.k, self.nbytes = alloc, 0, None, 0, 0

    def _prepare(self):
        nb = {e.shard_message_bytes() for e in self.es}
        assert len(nb) == 1, "ranks disagree on the message size: %r" % (nb,)
        self.nbytes = nb.pop()
        if self.nbytes > self.max_bytes:
            self.max_bytes = self.nbytes
            self.msgs = [[self._alloc(self.max_bytes) for _ in range(self.G)] for _ in range(2)]

    def load_carriers(self, xyz):
        for e in self.es:
            e.load_carriers(xyz)
        self.refresh()

    def refresh(self):
        sts = [e.state() for e in self.es]
        assert len({(s["step"], s["n_active"]) for s in sts}) == 1, "ranks diverged"
        self._prepare()
        return sts[0]

    def step(self, n=1):
        if self.msgs is None:
            self._prepare()
        for _ in range(int(n)):
            msgs = self.msgs[self.k & 1]
            self.k += 1
            for e, m in zip(self.es, msgs):
                e.shard_local(m.data_ptr(), self.nbytes)
            ptrs = [m.data_ptr() for m in msgs]
            for e in self.es:
                e.shard_commit(ptrs, self.nbytes)

    def run_to_collection(self, max_steps=10 ** 9):
        st = self.refresh()
        step0, done = st["step"], 0
        while st["n_active"] > 0 and done < max_steps:
            self.step(min(REFRESH_STEPS, max_steps - done))
            st = self.refresh()
            done = st["step"] - step0
        return done, st["n_active"]

    def totals(self):
        sts = [e.state() for e in self.es]
        out = dict(sts[0])
        for k in ("n_collected", "n_out_of_window", "pair_interactions"):
            out[k] = sum(s[k] for s in sts)
        return out

    def image(self):
        return sum(np.asarray(e.read_image()[0], dtype=np.int64) for e in self.es).astype(np.uint32)

    def last_messages(self):
        """The G messages of the most recent step (uint8 tensors), for tests."""
        return [m[: self.nbytes] for m in self.msgs[(self.k - 1) & 1]]
