"""CPU oracle (TEST INFRASTRUCTURE): ctypes wrapper around oracle/oracle.c.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It imports nothing from paper_2606_01547_b200.

Definitions: SURVEY.md §8(c) G, E, S, H, T, R, B, P, following PAPER.md:55 (three steps)
and the profile names of PAPER.md:80, :85, :87, :103.  All arithmetic is float64 in
oracle.c; this file only marshals numpy arrays.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.c")
_LIB_PATH = os.path.join(_HERE, "liboracle.so")
_lib = None

_d = ctypes.c_double
_i = ctypes.c_int
_i64 = ctypes.c_int64
_dp = ctypes.POINTER(ctypes.c_double)


def build(force=False):
    """Compile oracle.c -> liboracle.so with gcc (-O2, no fast-math; OpenMP on the outer loops only)."""
    srcs = [_SRC, os.path.join(os.path.dirname(_SRC), "oracle_next.c")]
    if (not force and os.path.exists(_LIB_PATH)
            and all(os.path.getmtime(_LIB_PATH) >= os.path.getmtime(f) for f in srcs)):
        return _LIB_PATH
    cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
           "-o", _LIB_PATH] + srcs + ["-lm"]
    subprocess.run(cmd, check=True)
    return _LIB_PATH


def _ptr(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _arr(a, shape=None):
    if a is None:
        return None
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None:
        a = a.reshape(shape)
    return a


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB_PATH)
        L.orc_set_threads.argtypes = [_i]
        L.orc_get_max_threads.restype = _i
        L.orc_grid.argtypes = [_i, _i, _d, _d, _d, _i, _dp, _dp]
        L.orc_ellipticity.argtypes = [_d, _d, _dp, _dp]
        L.orc_sie_alpha.argtypes = [_d, _d, _dp, _dp, _dp]
        L.orc_sie_kappa.argtypes = [_d, _d, _dp]
        L.orc_sie_kappa.restype = _d
        L.orc_shear_alpha.argtypes = [_d, _d, _d, _d, _dp, _dp]
        L.orc_pointmass_alpha.argtypes = [_d, _d, _d, _d, _d, _dp, _dp]
        for name in ("orc_tnfw_F",):
            getattr(L, name).argtypes = [_d]
            getattr(L, name).restype = _d
        for name in ("orc_tnfw_L", "orc_tnfw_g", "orc_tnfw_g_closed", "orc_tnfw_g_series"):
            getattr(L, name).argtypes = [_d, _d]
            getattr(L, name).restype = _d
        L.orc_tnfw_alpha.argtypes = [_d, _d, _d, _d, _d, _d, _d, _dp, _dp]
        L.orc_tnfw_kappa.argtypes = [_d] * 7
        L.orc_tnfw_kappa.restype = _d
        L.orc_ray_shoot.argtypes = [_i64, _dp, _dp, _dp, _dp, _i64, _dp, _dp, _dp]
        L.orc_sersic.argtypes = [_d, _d, _dp]
        L.orc_sersic.restype = _d
        L.orc_source_brightness.argtypes = [_i64, _dp, _dp, _i, _dp, _dp]
        L.orc_bin.argtypes = [_i, _i, _i, _d, _dp, _dp]
        L.orc_convolve.argtypes = [_i, _i, _dp, _i, _i, _dp, _dp]
        L.orc_prepsf_rows.argtypes = [_i, _i, _d, _d, _d, _i, _dp, _dp, _i64, _dp, _i, _dp, _i, _i, _dp]
        L.orc_simulate_image.argtypes = [_i, _i, _d, _d, _d, _i, _dp, _dp, _i64, _dp, _i, _dp,
                                         _i, _i, _dp, _dp, _dp]
        L.orc_simulate_batch.argtypes = [_i64, _i, _i, _d, _d, _d, _i, _dp, _dp, _i64, _dp, _i, _dp,
                                         _i, _i, _dp, _dp]
        _i32p = ctypes.POINTER(ctypes.c_int32)
        L.orc_chi2_batch.argtypes = [_i64, _i64, _dp, _dp, _dp, _dp]
        L.orc_lensing_maps.argtypes = [_i64, _dp, _dp, _dp, _dp, _i64, _dp, _dp, _dp, _dp, _dp]
        L.orc_profile_alpha.argtypes = [_i, _dp, _d, _d, _dp, _dp]
        L.orc_profile_kappa.argtypes = [_i, _dp, _d, _d]
        L.orc_profile_kappa.restype = _d
        L.orc_ray_shoot_profiles.argtypes = [_i64, _dp, _dp, _i64, _i32p, _dp, _dp, _dp]
        L.orc_light.argtypes = [_i, _dp, _d, _d]
        L.orc_light.restype = _d
        L.orc_light_profiles.argtypes = [_i64, _dp, _dp, _i64, _i32p, _dp, _dp]
        L.orc_profile_alpha2.argtypes = [_i, _dp, _d, _d, _dp, _dp]
        L.orc_profile_kappa2.argtypes = [_i, _dp, _d, _d]
        L.orc_profile_kappa2.restype = _d
        L.orc_ray_shoot_profiles2.argtypes = [_i64, _dp, _dp, _i64, _i32p, _dp, _dp, _dp]
        L.orc_pjaffe_ell_potential.argtypes = [_d, _d, _dp]
        L.orc_pjaffe_ell_potential.restype = _d
        L.orc_multipole_potential.argtypes = [_d, _d, _dp]
        L.orc_multipole_potential.restype = _d
        L.orc_core_sersic_n.argtypes = [_i64, _dp, _dp, _dp, _d, _d, _dp]
        L.orc_shapelets_n.argtypes = [_i64, _dp, _dp, _i, _d, _d, _d, _dp, _dp]
        L.orc_convolve_supersampled.argtypes = [_i, _i, _i, _dp, _i, _i, _dp, _dp, _dp]
        _lib = L
    return _lib


def set_threads(n):
    lib().orc_set_threads(int(n))


def max_threads():
    return int(lib().orc_get_max_threads())


# ----------------------------------------------------------------- scalar functions
def ellipticity(e1, e2):
    phi, q = _d(), _d()
    lib().orc_ellipticity(e1, e2, ctypes.byref(phi), ctypes.byref(q))
    return phi.value, q.value


def sie_alpha(x, y, theta_E, e1, e2, cx=0.0, cy=0.0):
    p = (_d * 5)(theta_E, e1, e2, cx, cy)
    ax, ay = _d(), _d()
    lib().orc_sie_alpha(x, y, p, ctypes.byref(ax), ctypes.byref(ay))
    return ax.value, ay.value


def sie_kappa(x, y, theta_E, e1, e2, cx=0.0, cy=0.0):
    p = (_d * 5)(theta_E, e1, e2, cx, cy)
    return lib().orc_sie_kappa(x, y, p)


def shear_alpha(x, y, g1, g2):
    ax, ay = _d(), _d()
    lib().orc_shear_alpha(x, y, g1, g2, ctypes.byref(ax), ctypes.byref(ay))
    return ax.value, ay.value


def pointmass_alpha(x, y, theta_E, cx=0.0, cy=0.0):
    ax, ay = _d(), _d()
    lib().orc_pointmass_alpha(x, y, theta_E, cx, cy, ctypes.byref(ax), ctypes.byref(ay))
    return ax.value, ay.value


def tnfw_F(X):
    return lib().orc_tnfw_F(X)


def tnfw_L(X, tau):
    return lib().orc_tnfw_L(X, tau)


def tnfw_g(X, tau):
    return lib().orc_tnfw_g(X, tau)


def tnfw_g_closed(X, tau):
    return lib().orc_tnfw_g_closed(X, tau)


def tnfw_g_series(X, tau):
    return lib().orc_tnfw_g_series(X, tau)


def tnfw_alpha(x, y, cx, cy, Rs, alpha_Rs, r_trunc):
    ax, ay = _d(), _d()
    lib().orc_tnfw_alpha(x, y, cx, cy, Rs, alpha_Rs, r_trunc, ctypes.byref(ax), ctypes.byref(ay))
    return ax.value, ay.value


def tnfw_kappa(x, y, cx, cy, Rs, alpha_Rs, r_trunc):
    return lib().orc_tnfw_kappa(x, y, cx, cy, Rs, alpha_Rs, r_trunc)


def sersic(x, y, amp, R_sersic, n_sersic, e1, e2, cx, cy):
    p = (_d * 7)(amp, R_sersic, n_sersic, e1, e2, cx, cy)
    return lib().orc_sersic(x, y, p)


# ----------------------------------------------------------------- array functions
def grid(nx, ny, pixel_scale, cx=0.0, cy=0.0, supersample=1):
    n = nx * supersample * ny * supersample
    tx = np.empty(n)
    ty = np.empty(n)
    lib().orc_grid(nx, ny, pixel_scale, cx, cy, supersample, _ptr(tx), _ptr(ty))
    return tx, ty


def _lens_args(sie, shear, tnfw):
    sie = _arr(sie)
    shear = _arr(shear)
    if tnfw is None:
        tnfw = np.zeros((5, 0))
    tnfw = _arr(tnfw)
    assert tnfw.ndim == 2 and tnfw.shape[0] == 5
    return sie, shear, tnfw


def ray_shoot(theta_x, theta_y, sie=None, shear=None, tnfw=None):
    tx = _arr(theta_x).ravel()
    ty = _arr(theta_y).ravel()
    sie, shear, tnfw = _lens_args(sie, shear, tnfw)
    bx = np.empty_like(tx)
    by = np.empty_like(ty)
    lib().orc_ray_shoot(tx.size, _ptr(tx), _ptr(ty), _ptr(sie), _ptr(shear), tnfw.shape[1], _ptr(tnfw),
                        _ptr(bx), _ptr(by))
    return bx, by


def source_brightness(beta_x, beta_y, sources):
    bx = _arr(beta_x).ravel()
    by = _arr(beta_y).ravel()
    src = _arr(sources).reshape(-1, 7)
    out = np.empty_like(bx)
    lib().orc_source_brightness(bx.size, _ptr(bx), _ptr(by), src.shape[0], _ptr(src), _ptr(out))
    return out


def bin_rays(nx, ny, supersample, pixel_scale, flux):
    f = _arr(flux).ravel()
    assert f.size == nx * ny * supersample * supersample
    img = np.empty((ny, nx))
    lib().orc_bin(nx, ny, supersample, pixel_scale, _ptr(f), _ptr(img))
    return img


def convolve(image, kernel):
    img = _arr(image)
    ker = _arr(kernel)
    out = np.empty_like(img)
    lib().orc_convolve(img.shape[0], img.shape[1], _ptr(img), ker.shape[0], ker.shape[1], _ptr(ker), _ptr(out))
    return out


def prepsf_rows(w, j0=0, j1=None):
    """Pre-PSF image rows [j0, j1) of a workloads.Workload-like object (duck-typed; no import)."""
    j1 = w.ny if j1 is None else j1
    sie, shear, tnfw = _lens_args(w.sie, w.shear, w.tnfw)
    src = _arr(w.sources).reshape(-1, 7)
    out = np.empty((j1 - j0, w.nx))
    lib().orc_prepsf_rows(w.nx, w.ny, w.pixel_scale, w.cx, w.cy, w.supersample, _ptr(sie), _ptr(shear),
                          tnfw.shape[1], _ptr(tnfw), src.shape[0], _ptr(src), j0, j1, _ptr(out))
    return out


def prepsf_pixels(w, j, cols):
    """Pre-PSF values of the pixels (j, i), i in cols, by composing the oracle's steps on just their sub-rays:
    definition G for the s x s sub-ray angles, orc_ray_shoot, orc_source_brightness, definition B.
    Used to sample configs whose full image would take core-hours."""
    s = int(w.supersample)
    cols = np.asarray(cols, dtype=np.int64)
    NX, NY = w.nx * s, w.ny * s
    h = w.pixel_scale / s
    shape = (len(cols), s, s)                                                            # [pixel][sub-row][sub-column]
    I = np.broadcast_to(cols[:, None, None] * s + np.arange(s)[None, None, :], shape).astype(np.float64)
    J = np.broadcast_to(j * s + np.arange(s)[None, :, None], shape).astype(np.float64)
    tx = w.cx + (I - 0.5 * (NX - 1)) * h
    ty = w.cy + (J - 0.5 * (NY - 1)) * h
    bx, by = ray_shoot(tx.ravel(), ty.ravel(), w.sie, w.shear, w.tnfw)
    flux = source_brightness(bx, by, w.sources).reshape(len(cols), s * s)
    return w.pixel_scale ** 2 * flux.sum(axis=1) / float(s * s)


def simulate_image(w):
    """Whole pipeline on one system; returns (pre_psf, image)."""
    sie, shear, tnfw = _lens_args(w.sie, w.shear, w.tnfw)
    src = _arr(w.sources).reshape(-1, 7)
    psf = _arr(w.psf)
    pre = np.empty((w.ny, w.nx))
    out = np.empty((w.ny, w.nx))
    lib().orc_simulate_image(w.nx, w.ny, w.pixel_scale, w.cx, w.cy, w.supersample, _ptr(sie), _ptr(shear),
                             tnfw.shape[1], _ptr(tnfw), src.shape[0], _ptr(src),
                             psf.shape[0], psf.shape[1], _ptr(psf), _ptr(pre), _ptr(out))
    return pre, out


def simulate_batch(bw, systems=None):
    """Batched pipeline; `systems` optionally selects a subset of system indices."""
    idx = np.arange(bw.B) if systems is None else np.asarray(systems)
    sie = _arr(bw.sie[idx])
    shear = _arr(bw.shear[idx])
    tnfw = _arr(bw.tnfw[idx])
    src = _arr(bw.sources[idx])
    psf = _arr(bw.psf[idx])
    out = np.empty((idx.size, bw.ny, bw.nx))
    lib().orc_simulate_batch(idx.size, bw.nx, bw.ny, bw.pixel_scale, bw.cx, bw.cy, bw.supersample,
                             _ptr(sie), _ptr(shear), tnfw.shape[2], _ptr(tnfw), src.shape[1], _ptr(src),
                             psf.shape[1], psf.shape[2], _ptr(psf), _ptr(out))
    return out


def chi2_batch(models, data, sigma):
    """chi2[b] = sum_pixels ((models[b] - data) / sigma)^2 (reading Q24; PAPER.md:120-126 swarm inner loop)."""
    m = _arr(models)
    d = _arr(data)
    sg = _arr(sigma)
    m = m.reshape(-1, d.size)
    out = np.empty(m.shape[0])
    lib().orc_chi2_batch(m.shape[0], d.size, _ptr(m), _ptr(d), _ptr(sg), _ptr(out))
    return out


# ------------------------------------------------------------------ SURVEY section 8(f) rows (oracle_next.c)
DEFLECTOR_TYPES = {"CONVERGENCE": 0, "SIS": 1, "NFW": 2, "HERNQUIST": 3, "PJAFFE": 4, "SIE": 5, "SHEAR": 6, "TNFW": 7,
                   "NIE": 8, "EPL": 9, "MULTIPOLE": 10, "CSE": 11, "PJAFFE_ELLIPSE_POTENTIAL": 12}
LIGHT_TYPES = {"SERSIC_ELLIPSE": 0, "GAUSSIAN_ELLIPSE": 1}


def _typed(records, table):
    """[(name, [params...]), ...] -> (int32 types [n], float64 params [n][8])"""
    types = np.array([table[name] for name, _ in records], dtype=np.int32)
    params = np.zeros((len(records), 8))
    for k, (_, p) in enumerate(records):
        params[k, :len(p)] = p
    return types, params


def lensing_maps(theta_x, theta_y, sie=None, shear=None, tnfw=None):
    """(kappa, gamma1, gamma2, mu) of SIE + shear + TNFW at the given points (NEXT-2)."""
    tx = _arr(theta_x).ravel()
    ty = _arr(theta_y).ravel()
    sie_a, shear_a, tn = _lens_args(sie, shear, tnfw)
    out = [np.empty_like(tx) for _ in range(4)]
    lib().orc_lensing_maps(tx.size, _ptr(tx), _ptr(ty), _ptr(sie_a), _ptr(shear_a), tn.shape[1], _ptr(tn),
                           *[_ptr(o) for o in out])
    return tuple(out)


def profile_alpha(name, params, x, y):
    p = np.zeros(8)
    p[:len(params)] = params
    ax, ay = ctypes.c_double(), ctypes.c_double()
    lib().orc_profile_alpha2(DEFLECTOR_TYPES[name], _ptr(p), float(x), float(y), ctypes.byref(ax), ctypes.byref(ay))
    return ax.value, ay.value


def profile_kappa(name, params, x, y):
    p = np.zeros(8)
    p[:len(params)] = params
    return lib().orc_profile_kappa2(DEFLECTOR_TYPES[name], _ptr(p), float(x), float(y))


def ray_shoot_profiles(theta_x, theta_y, deflectors):
    """beta = theta - sum of the typed deflectors [(name, params), ...] (NEXT-1)."""
    tx = _arr(theta_x).ravel()
    ty = _arr(theta_y).ravel()
    types, params = _typed(deflectors, DEFLECTOR_TYPES)
    bx, by = np.empty_like(tx), np.empty_like(ty)
    lib().orc_ray_shoot_profiles2(tx.size, _ptr(tx), _ptr(ty), len(types), types.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)),
                                 _ptr(params), _ptr(bx), _ptr(by))
    return bx, by


def light(name, params, x, y):
    p = np.zeros(8)
    p[:len(params)] = params
    return lib().orc_light(LIGHT_TYPES[name], _ptr(p), float(x), float(y))


def light_profiles(beta_x, beta_y, components):
    """sum of typed light components [(name, params), ...] at (beta_x, beta_y) (NEXT-1)."""
    bx = _arr(beta_x).ravel()
    by = _arr(beta_y).ravel()
    types, params = _typed(components, LIGHT_TYPES)
    out = np.empty_like(bx)
    lib().orc_light_profiles(bx.size, _ptr(bx), _ptr(by), len(types), types.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)),
                             _ptr(params), _ptr(out))
    return out



def core_sersic(beta_x, beta_y, amp, R_sersic, n_sersic, Rb, gamma, alpha, e1, e2, cx, cy):
    """CORE_SERSIC surface brightness (reading Q33) at (beta_x, beta_y)."""
    bx = _arr(beta_x).ravel()
    by = _arr(beta_y).ravel()
    p = np.array([amp, R_sersic, n_sersic, Rb, gamma, alpha, e1, e2], dtype=np.float64)
    out = np.empty_like(bx)
    lib().orc_core_sersic_n(bx.size, _ptr(bx), _ptr(by), _ptr(p), float(cx), float(cy), _ptr(out))
    return out


def shapelet_count(n_max):
    return (n_max + 1) * (n_max + 2) // 2


def shapelets(beta_x, beta_y, n_max, beta, cx, cy, coef):
    """SHAPELETS surface brightness (reading Q34): coefficients ordered by N = n1 + n2 ascending, n2 = 0 ... N."""
    bx = _arr(beta_x).ravel()
    by = _arr(beta_y).ravel()
    c = _arr(coef).ravel()
    assert c.size == shapelet_count(n_max)
    out = np.empty_like(bx)
    lib().orc_shapelets_n(bx.size, _ptr(bx), _ptr(by), int(n_max), float(beta), float(cx), float(cy), _ptr(c), _ptr(out))
    return out


def convolve_supersampled(rays, supersample, kernel_fine):
    """NEXT-4: unbinned ray image [ny s][nx s] (x) PSF on the ray grid, then s x s binning -> [ny][nx]."""
    r = _arr(rays)
    k = _arr(kernel_fine)
    s = int(supersample)
    NY, NX = r.shape
    ny, nx = NY // s, NX // s
    tmp = np.empty_like(r)
    out = np.empty((ny, nx))
    lib().orc_convolve_supersampled(ny, nx, s, _ptr(r), k.shape[0], k.shape[1], _ptr(k), _ptr(tmp), _ptr(out))
    return out


def multipole_potential(x, y, m, a_m, phi_m, cx=0.0, cy=0.0):
    p = np.array([m, a_m, phi_m, cx, cy, 0, 0, 0], dtype=np.float64)
    return lib().orc_multipole_potential(float(x), float(y), _ptr(p))


def pjaffe_ell_potential(x, y, sigma0, Ra, Rs, e1, e2, cx=0.0, cy=0.0):
    p = np.array([sigma0, Ra, Rs, e1, e2, cx, cy, 0], dtype=np.float64)
    return lib().orc_pjaffe_ell_potential(float(x), float(y), _ptr(p))
