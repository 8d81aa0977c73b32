"""Test infrastructure: a CPU "engine" with the interface paper_2203_11043_b200/sharded.py drives (set_shard,
shard_message_bytes, shard_local, shard_commit, state, read_image), whose arithmetic is the FP64 oracle's
(goracle_coulomb_field on the share's targets against all sources + goracle_advance per carrier, FP32 state).
It lets the world_size-2 gloo test run the product's host orchestration — message sizing, the all-gather of
variable-length shares, commit order, the integer reductions — on CPU, and produces byte-identical message layouts
to the CUDA kernels' (header | x[] | y[] | z[] | id[]), so GPU messages can be checked against it too."""
import ctypes as C

import numpy as np

from oracle import goracle as g

HEADER = 256


def _bucket(t):
    b = 1
    while b < t:
        b <<= 1
    return b


def share_of(n, rank, world):
    T = (n + 255) // 256
    a, b = (T * rank // world) * 256, (T * (rank + 1) // world) * 256
    lo, hi = min(a, n), min(b, n)
    return lo, hi - lo


def _view(ptr, nbytes):
    return np.ctypeslib.as_array((C.c_uint8 * int(nbytes)).from_address(int(ptr)))


class OracleShardEngine:
    def __init__(self, params, P):
        """params: goracle Params; P: the workload's parameter dict (image window, pitch, z_well, softening, eps_si)."""
        self.params, self.P = params, P
        self.rank, self.world = 0, 1
        self.xyz = np.zeros((0, 3), dtype=np.float32)
        self.ids = np.zeros(0, dtype=np.uint32)
        self.step_index = 0
        self.n_loaded = self.n_collected = self.n_over = self.pairs = 0
        self.n_bound = 0
        self.image = np.zeros((P["img_ny"], P["img_nx"]), dtype=np.uint32)
        self.diverged = False

    def set_shard(self, rank, world):
        assert self.n_loaded == 0
        self.rank, self.world = rank, world

    def _bin(self, x, y):
        P = self.P
        ix = int(np.floor((float(x) - P["img_x0_um"]) / P["pixel_pitch_um"]))
        iy = int(np.floor((float(y) - P["img_y0_um"]) / P["pixel_pitch_um"]))
        self.n_collected += 1
        if 0 <= ix < P["img_nx"] and 0 <= iy < P["img_ny"]:
            self.image[iy, ix] += 1
        else:
            self.n_over += 1

    def load_carriers(self, xyz):
        a = np.ascontiguousarray(xyz, dtype=np.float32).reshape(-1, 3)
        ids = np.arange(self.n_loaded, self.n_loaded + len(a), dtype=np.uint32)
        keep = a[:, 2].astype(np.float64) > self.P["z_well_um"]
        if self.rank == 0:                                   # holes collected at load: binned by rank 0 only
            for r in a[~keep]:
                self._bin(r[0], r[1])
        self.xyz = np.concatenate([self.xyz, a[keep]])
        self.ids = np.concatenate([self.ids, ids[keep]])
        self.n_loaded += len(a)
        self.n_bound = len(self.ids)

    def state(self):
        self.n_bound = len(self.ids)
        if self.diverged:
            raise RuntimeError("ranks diverged")
        return dict(step=self.step_index, n_active=len(self.ids), n_loaded=self.n_loaded, n_collected=self.n_collected,
                    n_out_of_window=self.n_over, pair_interactions=self.pairs)

    def shard_message_bytes(self):
        tiles = _bucket(max(1, (max(self.n_bound, 1) + 255) // 256))
        return HEADER + 16 * 256 * ((tiles + self.world - 1) // self.world)

    def shard_local(self, ptr, nbytes):
        m = _view(ptr, nbytes)
        bs = (nbytes - HEADER) // 16 // 256 * 256
        n = len(self.ids)
        t0, nt = share_of(n, self.rank, self.world)
        assert nt <= bs
        out_xyz, out_ids = [], []
        if nt:
            E = g.coulomb_field(self.xyz.astype(np.float64), eps_um=self.P["softening_um"],
                                Kp=g.coulomb_constant(self.P["eps_si"]), targets=np.arange(t0, t0 + nt))
            for k in range(nt):
                i = t0 + k
                r_new, _ = g.advance(self.params, self.step_index, int(self.ids[i]), self.xyz[i].astype(np.float64), E[k])
                r32 = r_new.astype(np.float32)               # FP32 state
                if float(r32[2]) <= self.P["z_well_um"]:
                    self._bin(r32[0], r32[1])
                else:
                    out_xyz.append(r32)
                    out_ids.append(self.ids[i])
        c = len(out_ids)
        m[:HEADER] = 0
        m[:16].view(np.uint32)[:] = (c, nt, n, self.rank)
        m[16:24].view(np.uint64)[0] = self.step_index
        body = m[HEADER:HEADER + 16 * bs].view(np.uint32).reshape(4, bs)
        if c:
            body[:3, :c] = np.stack(out_xyz).T.copy().view(np.uint32)
            body[3, :c] = np.asarray(out_ids, dtype=np.uint32)
        self._nt = nt

    def shard_commit(self, ptrs, nbytes):
        assert len(ptrs) == self.world
        bs = (nbytes - HEADER) // 16 // 256 * 256
        xs, ids = [], []
        for r, p in enumerate(ptrs):
            m = _view(p, nbytes)
            c, nt, nb, rk = (int(v) for v in m[:16].view(np.uint32))
            st = int(m[16:24].view(np.uint64)[0])
            if nb != len(self.ids) or st != self.step_index or rk != r:
                self.diverged = True
            body = m[HEADER:HEADER + 16 * bs].view(np.uint32).reshape(4, bs)
            xs.append(body[:3, :c].copy().view(np.float32).T)
            ids.append(body[3, :c].copy())
        n = len(self.ids)
        self.pairs += self._nt * n
        if n:
            self.step_index += 1
        self.xyz = np.concatenate(xs).astype(np.float32).reshape(-1, 3)
        self.ids = np.concatenate(ids).astype(np.uint32)

    def read_image(self):
        return self.image.copy(), self.n_over

    def read_carriers(self):
        return self.xyz.copy(), self.ids.copy()
