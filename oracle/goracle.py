"""ctypes front end of the FP64 CPU oracle (oracle/goracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It imports nothing from
paper_2203_11043_b200 and shares no code with the CUDA path.

Argument marshalling only -- every number is computed in goracle.c.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "goracle.c")
_LIB = os.path.join(_HERE, "libgoracle.so")

COULOMB_OFF, DIFFUSION_OFF, DEPLETION_OFF, FP32_STATE = 1, 2, 4, 0x100


def build(force=False):
    """gcc -O2 -fopenmp oracle/goracle.c -> oracle/libgoracle.so (building the checker is not using it)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= max(os.path.getmtime(_SRC), os.path.getmtime(os.path.join(_HERE, "goracle.h")))):
        return _LIB
    cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
           "-ffp-contract=off", "-o", _LIB + ".tmp", _SRC, "-lm"]
    subprocess.run(cmd, check=True, cwd=_HERE)
    os.replace(_LIB + ".tmp", _LIB)
    return _LIB


class Params(C.Structure):
    _fields_ = [("T_K", C.c_double), ("a1_V_per_cm2", C.c_double), ("a2_V_per_cm", C.c_double),
                ("thickness_um", C.c_double), ("z_well_um", C.c_double), ("pixel_pitch_um", C.c_double),
                ("dt_ns", C.c_double), ("softening_um", C.c_double), ("eps_si", C.c_double),
                ("seed", C.c_uint64), ("img_nx", C.c_int32), ("img_ny", C.c_int32),
                ("img_x0_um", C.c_double), ("img_y0_um", C.c_double), ("flags", C.c_uint32), ("pad_", C.c_uint32)]


_lib = None


def lib():
    global _lib
    if _lib is not None:
        return _lib
    L = C.CDLL(build())
    dp, u32p, u64p = C.POINTER(C.c_double), C.POINTER(C.c_uint32), C.POINTER(C.c_uint64)
    L.goracle_depletion_field.restype = C.c_double
    L.goracle_depletion_field.argtypes = [C.c_double] * 3
    L.goracle_mobility.restype = C.c_double
    L.goracle_mobility.argtypes = [C.c_double] * 2
    L.goracle_thermal_voltage.restype = C.c_double
    L.goracle_thermal_voltage.argtypes = [C.c_double]
    L.goracle_diffusion_sigma.restype = C.c_double
    L.goracle_diffusion_sigma.argtypes = [C.c_double] * 3
    L.goracle_coulomb_constant.restype = C.c_double
    L.goracle_coulomb_constant.argtypes = [C.c_double]
    L.goracle_philox4x32_10.restype = None
    L.goracle_philox4x32_10.argtypes = [u32p, u32p, u32p]
    L.goracle_normals.restype = None
    L.goracle_normals.argtypes = [C.c_uint64, C.c_uint32, C.c_uint64, dp, u32p]
    L.goracle_xray_hole_count.restype = C.c_uint64
    L.goracle_xray_hole_count.argtypes = [C.c_double, C.c_double]
    L.goracle_xray_cloud.restype = None
    L.goracle_xray_cloud.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, dp, C.c_double, C.c_double, C.POINTER(C.c_float)]
    L.goracle_coulomb_field.restype = None
    L.goracle_coulomb_field.argtypes = [dp, dp, dp, C.c_uint64, u64p, C.c_uint64, C.c_double, C.c_double, dp, dp, dp]
    L.goracle_advance.restype = C.c_int
    L.goracle_advance.argtypes = [C.POINTER(Params), C.c_uint64, C.c_uint32, dp, dp, dp]
    L.goracle_create.restype = C.c_void_p
    L.goracle_create.argtypes = [C.POINTER(Params)]
    L.goracle_destroy.restype = None
    L.goracle_destroy.argtypes = [C.c_void_p]
    L.goracle_load.restype = C.c_int
    L.goracle_load.argtypes = [C.c_void_p, C.POINTER(C.c_float), C.c_uint64]
    L.goracle_load_state.restype = C.c_int
    L.goracle_load_state.argtypes = [C.c_void_p, dp, u32p, C.c_uint64, C.c_uint64]
    L.goracle_step.restype = C.c_uint64
    L.goracle_step.argtypes = [C.c_void_p, C.c_uint64]
    L.goracle_run.restype = C.c_uint64
    L.goracle_run.argtypes = [C.c_void_p, C.c_uint64]
    L.goracle_get_state.restype = None
    L.goracle_get_state.argtypes = [C.c_void_p, u64p, u64p, u64p, u64p, u64p]
    L.goracle_read_carriers.restype = C.c_uint64
    L.goracle_read_carriers.argtypes = [C.c_void_p, dp, u32p, C.c_uint64]
    L.goracle_read_image.restype = None
    L.goracle_read_image.argtypes = [C.c_void_p, u32p]
    L.goracle_read_collected.restype = C.c_uint64
    L.goracle_read_collected.argtypes = [C.c_void_p, dp, u64p, C.c_uint64]
    L.goracle_num_threads.restype = C.c_int
    L.goracle_num_threads.argtypes = []
    _lib = L
    return L


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def make_params(T_K=140.0, a1=2.81e4, a2=2.0e3, thickness_um=675.0, z_well_um=0.0, pixel_pitch_um=15.0,
                dt_ns=0.05, softening_um=1e-3, eps_si=11.7, seed=20220322, img_nx=64, img_ny=64,
                img_x0_um=-480.0, img_y0_um=-480.0, flags=0):
    return Params(T_K, a1, a2, thickness_um, z_well_um, pixel_pitch_um, dt_ns, softening_um, eps_si,
                  seed, img_nx, img_ny, img_x0_um, img_y0_um, flags, 0)


def depletion_field(z_um, a1, a2):
    return lib().goracle_depletion_field(z_um, a1, a2)


def mobility(E, T):
    return lib().goracle_mobility(float(E), float(T))


def thermal_voltage(T):
    return lib().goracle_thermal_voltage(float(T))


def diffusion_sigma(mu, T, dt_ns):
    return lib().goracle_diffusion_sigma(float(mu), float(T), float(dt_ns))


def coulomb_constant(eps_si=11.7):
    return lib().goracle_coulomb_constant(float(eps_si))


def xray_hole_count(E_e_eV, w_eV=3.77):
    """N = E_e / w_e (3.77 eV at 140 K), floored."""
    return int(lib().goracle_xray_hole_count(float(E_e_eV), float(w_eV)))


def xray_cloud(gen_seed, n, centre_um, sigma_um, thickness_um=675.0, first_index=0):
    """seeded 3-D Gaussian initial cloud, float32 (n,3)."""
    out = np.empty((int(n), 3), dtype=np.float32)
    c = np.ascontiguousarray(centre_um, dtype=np.float64)
    lib().goracle_xray_cloud(int(gen_seed), int(first_index), int(n), _dp(c), float(sigma_um), float(thickness_um),
                             out.ctypes.data_as(C.POINTER(C.c_float)))
    return out


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(v) & 0xffffffff for v in ctr])
    k = (C.c_uint32 * 2)(*[int(v) & 0xffffffff for v in key])
    o = (C.c_uint32 * 4)()
    lib().goracle_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def normals(seed, cid, step):
    n = np.zeros(3)
    w = (C.c_uint32 * 4)()
    lib().goracle_normals(int(seed), int(cid), int(step), _dp(n), w)
    return n, [int(v) for v in w]


def coulomb_field(xyz, eps_um=1e-3, Kp=None, targets=None):
    """E (V/cm) at targets (default: all) from all sources; xyz is (n,3), used as float64."""
    xyz = np.asarray(xyz, dtype=np.float64)
    n = xyz.shape[0]
    x, y, z = (np.ascontiguousarray(xyz[:, k]) for k in range(3))
    if Kp is None:
        Kp = coulomb_constant(11.7)
    if targets is None:
        m, tp = n, None
    else:
        t = np.ascontiguousarray(np.asarray(targets, dtype=np.uint64))
        m, tp = t.shape[0], t.ctypes.data_as(C.POINTER(C.c_uint64))
    E = [np.zeros(m) for _ in range(3)]
    lib().goracle_coulomb_field(_dp(x), _dp(y), _dp(z), n, tp, m, float(eps_um), float(Kp), _dp(E[0]), _dp(E[1]), _dp(E[2]))
    return np.stack(E, axis=1)


def advance(params, step, cid, r, Ecoul):
    r = np.ascontiguousarray(r, dtype=np.float64)
    e = np.ascontiguousarray(Ecoul, dtype=np.float64)
    out = np.zeros(3)
    c = lib().goracle_advance(C.byref(params), int(step), int(cid), _dp(r), _dp(e), _dp(out))
    return out, bool(c)


class Sim:
    """One event on the oracle: same call sequence as the C-ABI of the product."""

    def __init__(self, params):
        self.params = params
        self._h = lib().goracle_create(C.byref(params))
        if not self._h:
            raise ValueError("goracle_create: invalid parameters")

    def close(self):
        if self._h:
            lib().goracle_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def load(self, xyz_f32):
        a = np.ascontiguousarray(xyz_f32, dtype=np.float32).reshape(-1, 3)
        rc = lib().goracle_load(self._h, a.ctypes.data_as(C.POINTER(C.c_float)), a.shape[0])
        if rc != 0:
            raise ValueError("goracle_load: invalid carriers")

    def load_state(self, xyz, ids, step):
        a = np.ascontiguousarray(xyz, dtype=np.float64).reshape(-1, 3)
        i = np.ascontiguousarray(ids, dtype=np.uint32)
        lib().goracle_load_state(self._h, _dp(a), i.ctypes.data_as(C.POINTER(C.c_uint32)), a.shape[0], int(step))

    def step(self, n=1):
        return int(lib().goracle_step(self._h, int(n)))

    def run(self, max_steps=10 ** 9):
        return int(lib().goracle_run(self._h, int(max_steps)))

    def state(self):
        v = [C.c_uint64() for _ in range(5)]
        lib().goracle_get_state(self._h, *[C.byref(q) for q in v])
        return dict(zip(("step", "n_active", "n_collected", "n_out_of_window", "pair_interactions"),
                        (int(q.value) for q in v)))

    def carriers(self):
        n = int(lib().goracle_read_carriers(self._h, None, None, 0))
        xyz = np.zeros((n, 3))
        ids = np.zeros(n, dtype=np.uint32)
        lib().goracle_read_carriers(self._h, _dp(xyz), ids.ctypes.data_as(C.POINTER(C.c_uint32)), n)
        return xyz, ids

    def image(self):
        img = np.zeros((self.params.img_ny, self.params.img_nx), dtype=np.uint32)
        lib().goracle_read_image(self._h, img.ctypes.data_as(C.POINTER(C.c_uint32)))
        return img

    def collected(self):
        n = int(lib().goracle_read_collected(self._h, None, None, 0))
        xyz = np.zeros((n, 3))
        st = np.zeros(n, dtype=np.uint64)
        lib().goracle_read_collected(self._h, _dp(xyz), st.ctypes.data_as(C.POINTER(C.c_uint64)), n)
        return xyz, st


def num_threads():
    return int(lib().goracle_num_threads())
