"""Recorded experiment: can the three accumulates of eq. 6 move to
the tensor cores?  E_t = sum_s w_ts (r_s - r_t) is not a contraction — (r_s - r_t) depends on both indices — unless it is
expanded as  sum_s w_ts (r_s - c) - (r_t - c) sum_s w_ts  (c = centre of a 16-target mma tile), with W[targets x
sources] and [x y z 1][sources x 4] as the operands of mma.m16n8k8.  This test emulates that route on the CPU (TF32
operands split 3 ways = FP32-equivalent products, FP32 accumulators, the same 256-source two-level accumulation as
k_field) on the track geometry of config 3 and asserts the KILL CRITERION: the expanded form cancels catastrophically
(w reaches eps^-3 = 1e9 um^-3 for the closest pairs while |r_s - c| is hundreds of um on a track kept in load order), so
it misses the 1e-4 field tolerance by orders of magnitude where the present FP32 form (differences first) meets it with
a margin of 20.  No narrower arithmetic may reach the shipped path; this one does not even keep FP32's accuracy."""
import numpy as np

import workloads


def _tf32(x):
    b = np.asarray(x, dtype=np.float32).view(np.uint32).astype(np.uint64)
    return ((b + 0x1000) & 0xFFFFE000).astype(np.uint32).view(np.float32)


def _split3(x):
    parts, r = [], np.asarray(x, dtype=np.float32)
    for _ in range(3):
        h = _tf32(r)
        parts.append(h)
        r = (r - h).astype(np.float32)
    return parts


def test_tensor_core_form_of_eq6_fails_the_field_tolerance_on_track_geometry():
    w = workloads.make(3, n=65536)                       # 48 holes/um: a quarter of config 3's line density
    xyz = w["xyz"][w["xyz"][:, 2] > 0]
    n, eps2 = len(xyz), np.float32(1e-6)
    rng = np.random.default_rng(0)
    worst_present, worst_mma = 0.0, 0.0
    for t0 in rng.integers(0, n // 16, size=4) * 16:
        T = xyz[t0:t0 + 16]
        c = T.mean(axis=0).astype(np.float32)
        d = (xyz[None, :, :] - T[:, None, :]).astype(np.float32)
        r2 = (d[..., 0] * d[..., 0] + eps2).astype(np.float32)
        r2 = (d[..., 1] * d[..., 1] + r2).astype(np.float32)
        r2 = (d[..., 2] * d[..., 2] + r2).astype(np.float32)
        inv = (1.0 / np.sqrt(r2.astype(np.float64))).astype(np.float32)
        wts = (inv * inv * inv).astype(np.float32)
        ref = (wts.astype(np.float64)[..., None] * d.astype(np.float64)).sum(axis=1)
        acc = np.zeros((16, 3))
        for j in range(0, n, 256):                       # the shipped form: FP32 products of differences, tile partials
            acc += (wts[:, j:j + 256, None] * d[:, j:j + 256, :]).astype(np.float32).sum(axis=1, dtype=np.float32)
        worst_present = max(worst_present, float((np.linalg.norm(acc - ref, axis=1) / np.linalg.norm(ref, axis=1)).max()))
        B = np.concatenate([(xyz - c).astype(np.float32), np.ones((n, 1), np.float32)], axis=1)
        Wp, Bp = _split3(wts), _split3(B)
        out = np.zeros((16, 4))
        for j in range(0, n, 256):
            part = np.zeros((16, 4), dtype=np.float32)
            for a, wa in enumerate(Wp):
                for b, bb in enumerate(Bp):
                    if a + b < 3:
                        part = (part + (wa[:, j:j + 256].astype(np.float64) @ bb[j:j + 256].astype(np.float64)).astype(np.float32)).astype(np.float32)
            out += part
        E = out[:, :3] - (T - c).astype(np.float64) * out[:, 3:4]
        worst_mma = max(worst_mma, float((np.linalg.norm(E - ref, axis=1) / np.linalg.norm(ref, axis=1)).max()))
    print("eq. 6 on a track, max relative error of the field sum: shipped FP32 form %.2e, tensor-core (expanded) form %.2e"
          % (worst_present, worst_mma))
    assert worst_present < 1e-4 / 10
    assert worst_mma > 1e-4 * 100                        # the kill criterion, by more than two orders of magnitude
