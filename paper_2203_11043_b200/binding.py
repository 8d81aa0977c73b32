"""Thin Python binding of the C ABI in include/gcoreccd.h — argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind libgcoreccd.so.  PyTorch is used for what the
task allows it for: device memory (the handle's workspace is a torch uint8 tensor) and streams (the handle
runs on torch's current CUDA stream unless told otherwise).  There is no CPU fallback: loading fails loudly
if the library is missing, and gcoreccd_create fails without an sm_100 GPU.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

OK, MAX_STEPS = 0, 1
ERR_INVALID, ERR_STATE, ERR_CAPACITY, ERR_NOMEM, ERR_CUDA, ERR_NONFINITE = -1, -2, -3, -4, -5, -6
COULOMB_OFF, DIFFUSION_OFF, DEPLETION_OFF = 1, 2, 4

EXPORTS = ["gcoreccd_workspace_size", "gcoreccd_create", "gcoreccd_destroy", "gcoreccd_reset",
           "gcoreccd_load_carriers", "gcoreccd_load_snapshot", "gcoreccd_step", "gcoreccd_run_to_collection",
           "gcoreccd_read_image", "gcoreccd_get_state", "gcoreccd_read_carriers", "gcoreccd_read_collected", "gcoreccd_eval_field",
           "gcoreccd_load_events", "gcoreccd_run_events", "gcoreccd_get_events", "gcoreccd_read_event_carriers",
           "gcoreccd_xray_hole_count", "gcoreccd_generate_cloud", "gcoreccd_generate_xray_events",
           "gcoreccd_load_carriers_file", "gcoreccd_save_collected_file",
           "gcoreccd_set_farfield", "gcoreccd_farfield_stats",
           "gcoreccd_set_shard", "gcoreccd_shard_message_bytes", "gcoreccd_shard_local", "gcoreccd_shard_commit", "gcoreccd_set_shard_wait",
           "gcoreccd_profile_step", "gcoreccd_set_persistent", "gcoreccd_kernel_launches", "gcoreccd_debug_normals", "gcoreccd_debug_mobility", "gcoreccd_mobility_table_host", "gcoreccd_debug_microbench", "gcoreccd_strerror",
           "gcoreccd_field_noalloc", "gcoreccd_field_noalloc_error",
           "gcoreccd_last_error", "gcoreccd_version"]


class Params(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("flags", C.c_uint32), ("T_K", C.c_double),
                ("a1_V_per_cm2", C.c_double), ("a2_V_per_cm", C.c_double), ("thickness_um", C.c_double),
                ("z_well_um", C.c_double), ("pixel_pitch_um", C.c_double), ("dt_ns", C.c_double),
                ("softening_um", C.c_double), ("eps_si", C.c_double), ("seed", C.c_uint64),
                ("img_nx", C.c_int32), ("img_ny", C.c_int32), ("img_x0_um", C.c_double), ("img_y0_um", C.c_double),
                ("device", C.c_int32), ("reserved0", C.c_int32), ("stream", C.c_void_p), ("workspace", C.c_void_p),
                ("workspace_bytes", C.c_uint64), ("max_carriers", C.c_uint64)]


class GcoreccdError(RuntimeError):
    def __init__(self, code, what, detail=""):
        self.code = code
        super().__init__("%s failed: %s (%d)%s" % (what, strerror(code), code, (": " + detail) if detail else ""))


_lib = None


def library_path():
    return _build.LIB


def lib():
    """Load libgcoreccd.so (no build here: __graft_entry__.build() / `python -m paper_2203_11043_b200.build`)."""
    global _lib
    if _lib is not None:
        return _lib
    path = library_path()
    if not os.path.exists(path):
        raise RuntimeError("libgcoreccd.so is missing (%s): run `python -m paper_2203_11043_b200.build`; "
                           "there is no CPU fallback" % path)
    L = C.CDLL(path)
    vp, u64p, u32p, fp = C.c_void_p, C.POINTER(C.c_uint64), C.POINTER(C.c_uint32), C.POINTER(C.c_float)
    L.gcoreccd_workspace_size.restype = C.c_uint64
    L.gcoreccd_workspace_size.argtypes = [C.c_uint64, C.c_int32, C.c_int32]
    L.gcoreccd_create.restype = C.c_int
    L.gcoreccd_create.argtypes = [C.POINTER(Params), C.POINTER(vp)]
    L.gcoreccd_destroy.restype = C.c_int
    L.gcoreccd_destroy.argtypes = [vp]
    L.gcoreccd_reset.restype = C.c_int
    L.gcoreccd_reset.argtypes = [vp]
    L.gcoreccd_load_carriers.restype = C.c_int
    L.gcoreccd_load_carriers.argtypes = [vp, vp, C.c_uint64, C.c_int]
    L.gcoreccd_load_snapshot.restype = C.c_int
    L.gcoreccd_load_snapshot.argtypes = [vp, fp, u32p, C.c_uint64, C.c_uint64]
    L.gcoreccd_step.restype = C.c_int
    L.gcoreccd_step.argtypes = [vp, C.c_uint32]
    L.gcoreccd_run_to_collection.restype = C.c_int
    L.gcoreccd_run_to_collection.argtypes = [vp, C.c_uint64, u64p, u64p]
    L.gcoreccd_read_image.restype = C.c_int
    L.gcoreccd_read_image.argtypes = [vp, vp, C.c_uint64, u64p, C.c_int]
    L.gcoreccd_get_state.restype = C.c_int
    L.gcoreccd_get_state.argtypes = [vp, u64p, u64p, u64p, u64p, u64p, u64p]
    L.gcoreccd_read_carriers.restype = C.c_int
    L.gcoreccd_read_carriers.argtypes = [vp, vp, vp, C.c_uint64, u64p, C.c_int]
    L.gcoreccd_read_collected.restype = C.c_int
    L.gcoreccd_read_collected.argtypes = [vp, vp, vp, C.c_uint64, u64p]
    L.gcoreccd_eval_field.restype = C.c_int
    L.gcoreccd_eval_field.argtypes = [vp, vp, C.c_uint64, C.c_int]
    L.gcoreccd_load_events.restype = C.c_int
    L.gcoreccd_load_events.argtypes = [vp, vp, u64p, C.c_uint64, C.c_int]
    L.gcoreccd_run_events.restype = C.c_int
    L.gcoreccd_run_events.argtypes = [vp, C.c_uint64, u64p, u64p]
    L.gcoreccd_get_events.restype = C.c_int
    L.gcoreccd_get_events.argtypes = [vp, u64p, u64p, C.c_uint64, u64p]
    L.gcoreccd_read_event_carriers.restype = C.c_int
    L.gcoreccd_read_event_carriers.argtypes = [vp, C.c_uint64, vp, vp, C.c_uint64, u64p]
    dbl = C.POINTER(C.c_double)
    L.gcoreccd_xray_hole_count.restype = C.c_uint64
    L.gcoreccd_xray_hole_count.argtypes = [C.c_double, C.c_double]
    L.gcoreccd_generate_cloud.restype = C.c_int
    L.gcoreccd_generate_cloud.argtypes = [vp, C.c_uint64, dbl, C.c_double, C.c_uint64, C.c_uint64]
    L.gcoreccd_generate_xray_events.restype = C.c_int
    L.gcoreccd_generate_xray_events.argtypes = [vp, C.c_uint64, dbl, dbl, dbl, C.c_double, C.c_uint64, C.c_uint64, u64p]
    L.gcoreccd_load_carriers_file.restype = C.c_int
    L.gcoreccd_load_carriers_file.argtypes = [vp, C.c_char_p, u64p]
    L.gcoreccd_save_collected_file.restype = C.c_int
    L.gcoreccd_save_collected_file.argtypes = [vp, C.c_char_p, u64p]
    L.gcoreccd_set_shard.restype = C.c_int
    L.gcoreccd_set_shard.argtypes = [vp, C.c_uint32, C.c_uint32]
    L.gcoreccd_shard_message_bytes.restype = C.c_uint64
    L.gcoreccd_shard_message_bytes.argtypes = [vp]
    L.gcoreccd_shard_local.restype = C.c_int
    L.gcoreccd_shard_local.argtypes = [vp, vp, C.c_uint64]
    L.gcoreccd_shard_commit.restype = C.c_int
    L.gcoreccd_shard_commit.argtypes = [vp, C.POINTER(vp), C.c_uint32, C.c_uint64]
    L.gcoreccd_set_shard_wait.restype = C.c_int
    L.gcoreccd_set_shard_wait.argtypes = [vp, C.c_int]
    L.gcoreccd_set_farfield.restype = C.c_int
    L.gcoreccd_set_farfield.argtypes = [vp, C.c_double, C.c_uint32, C.c_uint64]
    L.gcoreccd_farfield_stats.restype = C.c_int
    L.gcoreccd_farfield_stats.argtypes = [vp, u64p, u64p, C.POINTER(C.c_double)]
    L.gcoreccd_profile_step.restype = C.c_int
    L.gcoreccd_profile_step.argtypes = [vp, fp]
    L.gcoreccd_set_persistent.restype = C.c_int
    L.gcoreccd_set_persistent.argtypes = [vp, C.c_int, C.c_uint64]
    L.gcoreccd_kernel_launches.restype = C.c_uint64
    L.gcoreccd_kernel_launches.argtypes = [vp]
    L.gcoreccd_debug_normals.restype = C.c_int
    L.gcoreccd_debug_normals.argtypes = [vp, u32p, u64p, C.c_uint64, C.POINTER(C.c_double), u32p]
    L.gcoreccd_debug_mobility.restype = C.c_int
    L.gcoreccd_debug_mobility.argtypes = [vp, C.POINTER(C.c_double), C.c_uint64, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    L.gcoreccd_mobility_table_host.restype = C.c_int
    L.gcoreccd_mobility_table_host.argtypes = [C.c_double, C.POINTER(C.c_double), C.c_uint64, C.POINTER(C.c_double)]
    L.gcoreccd_debug_microbench.restype = C.c_int
    L.gcoreccd_debug_microbench.argtypes = [C.c_int, C.c_uint32, C.c_uint32, C.POINTER(C.c_double)]
    L.gcoreccd_field_noalloc.restype = C.c_int
    L.gcoreccd_field_noalloc.argtypes = [vp, C.c_uint64, C.c_double, C.c_double, vp, vp]
    L.gcoreccd_field_noalloc_error.restype = C.c_char_p
    L.gcoreccd_field_noalloc_error.argtypes = []
    L.gcoreccd_strerror.restype = C.c_char_p
    L.gcoreccd_strerror.argtypes = [C.c_int]
    L.gcoreccd_last_error.restype = C.c_char_p
    L.gcoreccd_last_error.argtypes = [vp]
    L.gcoreccd_version.restype = C.c_char_p
    L.gcoreccd_version.argtypes = []
    _lib = L
    return L


def strerror(code):
    return lib().gcoreccd_strerror(int(code)).decode()


def version():
    return lib().gcoreccd_version().decode()


def xray_hole_count(E_e_eV, w_eV=3.77):
    return int(lib().gcoreccd_xray_hole_count(float(E_e_eV), float(w_eV)))


NOALLOC_MAX_CARRIERS = 16384


def field_noalloc(xyz_dev_ptr, n, softening_um, eps_si, out_dev_ptr, stream_handle=0):
    """include/gcoreccd.h gcoreccd_field_noalloc: eq. 6 for n <= NOALLOC_MAX_CARRIERS holes with no handle and no device
    allocation.  Device pointers (ints) in and out, enqueued on `stream_handle` (a cudaStream_t as int), not synchronised.
    All calls share one static scratch array: keep them on one stream."""
    rc = lib().gcoreccd_field_noalloc(C.c_void_p(int(xyz_dev_ptr)), int(n), float(softening_um), float(eps_si),
                                      C.c_void_p(int(out_dev_ptr)), C.c_void_p(int(stream_handle)))
    if rc != OK:
        raise GcoreccdError(rc, "gcoreccd_field_noalloc", lib().gcoreccd_field_noalloc_error().decode())


MICRO_KINDS = ["FFMA2 three distinct operands", "FFMA2 a*a+c", "FFMA2 shared operand", "FADD2", "FMUL2",
               "FFMA scalar three distinct", "FFMA scalar shared operand", "DFMA", "MUFU.RSQ", "eq. 6 mix (per packed instruction)",
               "F2F f64->f32", "F2F f32->f64", "DADD", "eq. 6 on the FP64 pipe (per interaction)",
               "eq. 6 mix, 8 packs + 1 FP64 target (per round)", "eq. 6 mix, 8 packs + 2 FP64 targets (per round)",
               "eq. 6 mix, 8 packs + 4 FP64 targets (per round)"]


def microbench(kind, iters=4096, warps_per_subpartition=2):
    """Cycles per warp-instruction per SM sub-partition (include/gcoreccd.h gcoreccd_debug_microbench)."""
    out = C.c_double()
    rc = lib().gcoreccd_debug_microbench(int(kind), int(iters), int(warps_per_subpartition), C.byref(out))
    if rc != OK:
        raise GcoreccdError(rc, "gcoreccd_debug_microbench")
    return float(out.value)


def mobility_table_host(T_K, E):
    """eq. 2 through the kernels' interpolation table, built and evaluated on the host (no GPU)."""
    e = np.ascontiguousarray(E, dtype=np.float64)
    out = np.zeros_like(e)
    dp = C.POINTER(C.c_double)
    rc = lib().gcoreccd_mobility_table_host(float(T_K), e.ctypes.data_as(dp), e.size, out.ctypes.data_as(dp))
    if rc != OK:
        raise GcoreccdError(rc, "gcoreccd_mobility_table_host")
    return out


def workspace_size(max_carriers, img_nx, img_ny):
    return int(lib().gcoreccd_workspace_size(int(max_carriers), int(img_nx), int(img_ny)))


class Gcoreccd:
    """One event on one GPU: gcoreccd_create / load_carriers / step / run_to_collection / read_image."""

    def __init__(self, max_carriers, T_K=140.0, a1=2.81e4, a2=2.0e3, thickness_um=675.0, z_well_um=0.0,
                 pixel_pitch_um=15.0, dt_ns=0.05, softening_um=1e-3, eps_si=11.7, seed=20220322,
                 img_nx=64, img_ny=64, img_x0_um=-480.0, img_y0_um=-480.0, flags=0, device=None, stream=None,
                 torch_workspace=True):
        import torch  # device memory and streams only

        L = lib()
        if not torch.cuda.is_available():
            raise RuntimeError("gcoreccd needs a CUDA device (sm_100a); there is no CPU fallback")
        self._torch = torch
        self.device = torch.cuda.current_device() if device is None else int(device)
        self._h = C.c_void_p()
        self.img_nx, self.img_ny = int(img_nx), int(img_ny)
        self.max_carriers = int(max_carriers)
        nbytes = workspace_size(max_carriers, img_nx, img_ny)
        if nbytes == 0:
            raise GcoreccdError(ERR_INVALID, "gcoreccd_workspace_size")
        self._ws = None
        ws_ptr = None
        if torch_workspace:
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda:%d" % self.device)
            ws_ptr = (self._ws.data_ptr() + 255) // 256 * 256
        if stream is None:
            stream = torch.cuda.current_stream(self.device)
            if stream.cuda_stream == 0:
                # the legacy default stream cannot be captured into CUDA graphs: give the handle its own torch stream
                stream = torch.cuda.Stream(self.device)
        self._stream = stream
        # handle 0 would read as "create your own" in the C ABI: name the legacy stream explicitly if asked for
        stream_handle = stream.cuda_stream if stream.cuda_stream else 1          # cudaStreamLegacy
        p = Params(C.sizeof(Params), int(flags), T_K, a1, a2, thickness_um, z_well_um, pixel_pitch_um, dt_ns,
                   softening_um, eps_si, int(seed), self.img_nx, self.img_ny, img_x0_um, img_y0_um, self.device, 0,
                   C.c_void_p(stream_handle), C.c_void_p(ws_ptr), nbytes if ws_ptr else 0, self.max_carriers)
        rc = L.gcoreccd_create(C.byref(p), C.byref(self._h))
        if rc != OK:
            self._h = C.c_void_p()
            raise GcoreccdError(rc, "gcoreccd_create")

    # ---- plumbing
    def _check(self, rc, what):
        if rc < 0:
            raise GcoreccdError(rc, what, lib().gcoreccd_last_error(self._h).decode())
        return rc

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            lib().gcoreccd_destroy(self._h)
            self._h = C.c_void_p()
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    # ---- the five calls of BASELINE.json:north_star
    def reset(self):
        self._check(lib().gcoreccd_reset(self._h), "gcoreccd_reset")

    def load_carriers(self, xyz):
        """xyz: (n,3) float32 numpy array (host) or torch CUDA tensor (device); copied."""
        torch = self._torch
        if isinstance(xyz, torch.Tensor):
            if xyz.device.type == "cuda":
                t = xyz.detach().to(torch.float32).contiguous().reshape(-1, 3)
                self._stream.wait_stream(torch.cuda.current_stream(self.device))   # producer of `t` may be another stream
                rc = lib().gcoreccd_load_carriers(self._h, C.c_void_p(t.data_ptr()), t.shape[0], 1)
                return self._check(rc, "gcoreccd_load_carriers")
            xyz = xyz.numpy()
        a = np.ascontiguousarray(xyz, dtype=np.float32).reshape(-1, 3)
        rc = lib().gcoreccd_load_carriers(self._h, C.c_void_p(a.ctypes.data), a.shape[0], 0)
        return self._check(rc, "gcoreccd_load_carriers")

    def load_carriers_ptr(self, host_ptr, n):
        """Host pointer variant (e.g. a pinned torch tensor's data_ptr())."""
        return self._check(lib().gcoreccd_load_carriers(self._h, C.c_void_p(int(host_ptr)), int(n), 0), "gcoreccd_load_carriers")

    def step(self, n=1):
        return self._check(lib().gcoreccd_step(self._h, int(n)), "gcoreccd_step")

    def run_to_collection(self, max_steps=10 ** 9):
        done, left = C.c_uint64(), C.c_uint64()
        rc = self._check(lib().gcoreccd_run_to_collection(self._h, int(max_steps), C.byref(done), C.byref(left)),
                         "gcoreccd_run_to_collection")
        return int(done.value), int(left.value), rc

    def read_image(self, device=False):
        over = C.c_uint64()
        if device:
            with self._torch.cuda.stream(self._stream):
                out = self._torch.empty((self.img_ny, self.img_nx), dtype=self._torch.int32, device="cuda:%d" % self.device)
            rc = lib().gcoreccd_read_image(self._h, C.c_void_p(out.data_ptr()), out.numel(), C.byref(over), 1)
        else:
            out = np.zeros((self.img_ny, self.img_nx), dtype=np.uint32)
            rc = lib().gcoreccd_read_image(self._h, C.c_void_p(out.ctypes.data), out.size, C.byref(over), 0)
        self._check(rc, "gcoreccd_read_image")
        return out, int(over.value)

    # ---- workload front end
    def generate_cloud(self, n, centre_um, sigma_um, gen_seed, first_index=0):
        c = (C.c_double * 3)(*[float(v) for v in centre_um])
        return self._check(lib().gcoreccd_generate_cloud(self._h, int(n), c, float(sigma_um), int(gen_seed), int(first_index)),
                           "gcoreccd_generate_cloud")

    def generate_xray_events(self, E_e_eV, centres_um, sigmas_um, gen_seed, w_eV=3.77, first_index=0):
        """Returns the hole count per event."""
        E = np.ascontiguousarray(E_e_eV, dtype=np.float64).reshape(-1)
        c = np.ascontiguousarray(centres_um, dtype=np.float64).reshape(-1, 3)
        sg = np.ascontiguousarray(sigmas_um, dtype=np.float64).reshape(-1)
        assert len(c) == len(E) == len(sg)
        counts = np.zeros(len(E), dtype=np.uint64)
        dbl = C.POINTER(C.c_double)
        rc = lib().gcoreccd_generate_xray_events(self._h, len(E), E.ctypes.data_as(dbl), c.ctypes.data_as(dbl), sg.ctypes.data_as(dbl),
                                                 float(w_eV), int(gen_seed), int(first_index),
                                                 counts.ctypes.data_as(C.POINTER(C.c_uint64)))
        self._check(rc, "gcoreccd_generate_xray_events")
        return counts

    def load_carriers_file(self, path):
        n = C.c_uint64()
        self._check(lib().gcoreccd_load_carriers_file(self._h, os.fsencode(path), C.byref(n)), "gcoreccd_load_carriers_file")
        return int(n.value)

    def save_collected_file(self, path):
        n = C.c_uint64()
        self._check(lib().gcoreccd_save_collected_file(self._h, os.fsencode(path), C.byref(n)), "gcoreccd_save_collected_file")
        return int(n.value)

    # ---- batched independent events (one thread block per event)
    def load_events(self, xyz, offsets):
        """xyz: (n,3) float32 numpy (host) or torch CUDA tensor; offsets: n_events+1 non-decreasing, offsets[0] = 0."""
        torch = self._torch
        off = np.ascontiguousarray(offsets, dtype=np.uint64)
        offp = off.ctypes.data_as(C.POINTER(C.c_uint64))
        if isinstance(xyz, torch.Tensor) and xyz.device.type == "cuda":
            t = xyz.detach().to(torch.float32).contiguous().reshape(-1, 3)
            self._stream.wait_stream(torch.cuda.current_stream(self.device))
            rc = lib().gcoreccd_load_events(self._h, C.c_void_p(t.data_ptr()), offp, len(off) - 1, 1)
        else:
            a = np.ascontiguousarray(xyz, dtype=np.float32).reshape(-1, 3)
            rc = lib().gcoreccd_load_events(self._h, C.c_void_p(a.ctypes.data), offp, len(off) - 1, 0)
        return self._check(rc, "gcoreccd_load_events")

    def load_events_ptr(self, host_ptr, offsets):
        off = np.ascontiguousarray(offsets, dtype=np.uint64)
        rc = lib().gcoreccd_load_events(self._h, C.c_void_p(int(host_ptr)), off.ctypes.data_as(C.POINTER(C.c_uint64)),
                                        len(off) - 1, 0)
        return self._check(rc, "gcoreccd_load_events")

    def run_events(self, max_steps=10 ** 9):
        ev, ca = C.c_uint64(), C.c_uint64()
        rc = self._check(lib().gcoreccd_run_events(self._h, int(max_steps), C.byref(ev), C.byref(ca)), "gcoreccd_run_events")
        return int(ev.value), int(ca.value), rc

    def events(self):
        n = C.c_uint64()
        self._check(lib().gcoreccd_get_events(self._h, None, None, 0, C.byref(n)), "gcoreccd_get_events")
        k = int(n.value)
        act = np.zeros(k, dtype=np.uint64)
        stp = np.zeros(k, dtype=np.uint64)
        self._check(lib().gcoreccd_get_events(self._h, act.ctypes.data_as(C.POINTER(C.c_uint64)),
                                              stp.ctypes.data_as(C.POINTER(C.c_uint64)), k, C.byref(n)), "gcoreccd_get_events")
        return act, stp

    def read_event_carriers(self, event):
        n = C.c_uint64()
        self._check(lib().gcoreccd_read_event_carriers(self._h, int(event), None, None, 0, C.byref(n)),
                    "gcoreccd_read_event_carriers")
        k = int(n.value)
        xyz = np.zeros((k, 3), dtype=np.float32)
        ids = np.zeros(k, dtype=np.uint32)
        if k:
            self._check(lib().gcoreccd_read_event_carriers(self._h, int(event), C.c_void_p(xyz.ctypes.data),
                                                           C.c_void_p(ids.ctypes.data), k, C.byref(n)),
                        "gcoreccd_read_event_carriers")
        return xyz, ids

    # ---- introspection / test hooks
    def state(self):
        v = [C.c_uint64() for _ in range(6)]
        self._check(lib().gcoreccd_get_state(self._h, *[C.byref(q) for q in v]), "gcoreccd_get_state")
        return dict(zip(("step", "n_active", "n_loaded", "n_collected", "n_out_of_window", "pair_interactions"),
                        (int(q.value) for q in v)))

    def read_carriers(self):
        n = C.c_uint64()
        self._check(lib().gcoreccd_read_carriers(self._h, None, None, 0, C.byref(n), 0), "gcoreccd_read_carriers")
        k = int(n.value)
        xyz = np.zeros((k, 3), dtype=np.float32)
        ids = np.zeros(k, dtype=np.uint32)
        if k:
            self._check(lib().gcoreccd_read_carriers(self._h, C.c_void_p(xyz.ctypes.data), C.c_void_p(ids.ctypes.data),
                                                     k, C.byref(n), 0), "gcoreccd_read_carriers")
        return xyz, ids

    def read_collected(self):
        """(xyz float32 (n,3), step uint32 (n,)) indexed by carrier id; NaN / 0xFFFFFFFF while still drifting."""
        n = C.c_uint64()
        self._check(lib().gcoreccd_read_collected(self._h, None, None, 0, C.byref(n)), "gcoreccd_read_collected")
        k = int(n.value)
        xyz = np.zeros((k, 3), dtype=np.float32)
        st = np.zeros(k, dtype=np.uint32)
        if k:
            self._check(lib().gcoreccd_read_collected(self._h, C.c_void_p(xyz.ctypes.data), C.c_void_p(st.ctypes.data), k,
                                                      C.byref(n)), "gcoreccd_read_collected")
        return xyz, st

    def read_carriers_into(self, host_ptr_xyz, cap):
        n = C.c_uint64()
        self._check(lib().gcoreccd_read_carriers(self._h, C.c_void_p(int(host_ptr_xyz)), None, int(cap), C.byref(n), 0),
                    "gcoreccd_read_carriers")
        return int(n.value)

    def load_snapshot(self, xyz, ids, step):
        a = np.ascontiguousarray(xyz, dtype=np.float32).reshape(-1, 3)
        i = np.ascontiguousarray(ids, dtype=np.uint32)
        rc = lib().gcoreccd_load_snapshot(self._h, a.ctypes.data_as(C.POINTER(C.c_float)),
                                          i.ctypes.data_as(C.POINTER(C.c_uint32)), a.shape[0], int(step))
        return self._check(rc, "gcoreccd_load_snapshot")

    def eval_field(self):
        k = self.state()["n_active"]
        E = np.zeros((k, 3), dtype=np.float32)
        if k:
            self._check(lib().gcoreccd_eval_field(self._h, C.c_void_p(E.ctypes.data), k, 0), "gcoreccd_eval_field")
        return E

    # ---- far-field variant (include/gcoreccd.h "Far-field approximation")
    def set_farfield(self, theta, resort_every=0, min_active=0):
        self._check(lib().gcoreccd_set_farfield(self._h, float(theta), int(resort_every), int(min_active)), "set_farfield")

    def farfield_stats(self):
        a, b, B = C.c_uint64(), C.c_uint64(), C.c_double()
        self._check(lib().gcoreccd_farfield_stats(self._h, C.byref(a), C.byref(b), C.byref(B)), "farfield_stats")
        return {"far_evals": int(a.value), "near_evals": int(b.value), "bound_B": float(B.value)}

    # ---- target sharding (include/gcoreccd.h "Target sharding"; the orchestration is sharded.py) ----
    def set_shard(self, rank, world):
        self._check(lib().gcoreccd_set_shard(self._h, int(rank), int(world)), "set_shard")

    def shard_message_bytes(self):
        return int(lib().gcoreccd_shard_message_bytes(self._h))

    def shard_local(self, msg_ptr, msg_bytes):
        self._check(lib().gcoreccd_shard_local(self._h, C.c_void_p(int(msg_ptr)), int(msg_bytes)), "shard_local")

    def shard_commit(self, msg_ptrs, msg_bytes):
        arr = (C.c_void_p * len(msg_ptrs))(*[int(p) for p in msg_ptrs])
        self._check(lib().gcoreccd_shard_commit(self._h, arr, len(msg_ptrs), int(msg_bytes)), "shard_commit")

    def set_shard_wait(self, on=True):
        self._check(lib().gcoreccd_set_shard_wait(self._h, int(bool(on))), "set_shard_wait")

    def profile_step(self):
        ms = (C.c_float * 4)()
        self._check(lib().gcoreccd_profile_step(self._h, ms), "gcoreccd_profile_step")
        return dict(field=float(ms[0]), advance=float(ms[1]), step=float(ms[3]))

    def set_persistent(self, on=True, max_active=0):
        mode = on if (isinstance(on, int) and not isinstance(on, bool)) else int(bool(on))   # 2: the CTA-tile kernels only
        self._check(lib().gcoreccd_set_persistent(self._h, int(mode), int(max_active)), "gcoreccd_set_persistent")

    def kernel_launches(self):
        return int(lib().gcoreccd_kernel_launches(self._h))

    def debug_normals(self, ids, steps):
        i = np.ascontiguousarray(ids, dtype=np.uint32)
        s = np.ascontiguousarray(steps, dtype=np.uint64)
        out = np.zeros((i.shape[0], 3), dtype=np.float64)
        w = np.zeros((i.shape[0], 4), dtype=np.uint32)
        rc = lib().gcoreccd_debug_normals(self._h, i.ctypes.data_as(C.POINTER(C.c_uint32)),
                                          s.ctypes.data_as(C.POINTER(C.c_uint64)), i.shape[0],
                                          out.ctypes.data_as(C.POINTER(C.c_double)), w.ctypes.data_as(C.POINTER(C.c_uint32)))
        self._check(rc, "gcoreccd_debug_normals")
        return out, w

    def debug_mobility(self, E):
        """(mu by the kernels' table, mu by the direct exp/log form) at field magnitudes E (V/cm)."""
        e = np.ascontiguousarray(E, dtype=np.float64)
        a, b = np.zeros_like(e), np.zeros_like(e)
        dp = C.POINTER(C.c_double)
        self._check(lib().gcoreccd_debug_mobility(self._h, e.ctypes.data_as(dp), e.size, a.ctypes.data_as(dp), b.ctypes.data_as(dp)),
                    "gcoreccd_debug_mobility")
        return a, b

    def synchronize(self):
        self._stream.synchronize()


def from_workload(w, flags=0, max_carriers=None, **kw):
    """Handle configured with a workloads.make() parameter set."""
    P = w["params"]
    return Gcoreccd(max_carriers or len(w["xyz"]), T_K=P["T_K"], a1=P["a1"], a2=P["a2"], thickness_um=P["thickness_um"],
                    z_well_um=P["z_well_um"], pixel_pitch_um=P["pixel_pitch_um"], dt_ns=P["dt_ns"],
                    softening_um=P["softening_um"], eps_si=P["eps_si"], seed=P["seed"], img_nx=P["img_nx"],
                    img_ny=P["img_ny"], img_x0_um=P["img_x0_um"], img_y0_um=P["img_y0_um"], flags=flags, **kw)
