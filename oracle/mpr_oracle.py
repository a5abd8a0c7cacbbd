"""ctypes wrapper of the CPU oracle (oracle/mpr_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke()
and bench.py's cpu_baseline / --impl reference legs may import this module.
It imports nothing from paper_1811_01604_b200.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mpr_oracle.c")
# Storage type of data and state: float32 (the configurations; the paper's Table 3) in this module; the module
# oracle.mpr_oracle64 executes this same file with _F64 set: -DORC_F64, float64 (the paper's Table 2; NEXT-3)
_F64 = bool(globals().get("_F64", False))
REAL = np.float64 if _F64 else np.float32
_CREAL = C.c_double if _F64 else C.c_float
_LIB = os.path.join(_HERE, "libmpr_oracle64.so" if _F64 else "libmpr_oracle.so")

TWO_PI_F = float(REAL(2.0 * np.pi))   # float32: 6.2831854820251465; float64: 6.283185307179586


def build(force: bool = False) -> str:
    """gcc -O2, no FMA contraction, no fast-math; OpenMP over one colour's rows."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
               "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"] + (["-DORC_F64"] if _F64 else [])
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        f32p = np.ctypeslib.ndpointer(REAL, flags="C_CONTIGUOUS")     # the storage type
        f64p = np.ctypeslib.ndpointer(np.float64, flags="C_CONTIGUOUS")
        u8p = np.ctypeslib.ndpointer(np.uint8, flags="C_CONTIGUOUS")
        u32p = np.ctypeslib.ndpointer(np.uint32, flags="C_CONTIGUOUS")
        L.orc_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.orc_philox4x32_10.restype = None
        L.orc_u01.argtypes = [C.c_uint32]
        L.orc_u01.restype = C.c_double
        L.orc_minmax.argtypes = [f32p, u8p, C.c_int64, C.POINTER(_CREAL), C.POINTER(_CREAL)]
        L.orc_minmax.restype = C.c_int64
        L.orc_eq1.argtypes = [_CREAL, _CREAL, _CREAL]
        L.orc_eq1.restype = _CREAL
        L.orc_transform.argtypes = [f32p, u8p, C.c_int, C.c_int, C.c_uint64, C.c_uint32,
                                    _CREAL, _CREAL, f32p]
        L.orc_transform.restype = None
        L.orc_local_energy.argtypes = [C.c_double] * 4
        L.orc_local_energy.restype = C.c_double
        L.orc_or_reflect.argtypes = [C.c_double] * 6 + [C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_double)]
        L.orc_or_reflect.restype = C.c_double
        L.orc_sweep.argtypes = [f32p, u8p, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                C.c_uint64, C.c_uint32, C.c_uint32, C.c_int,
                                C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_sweep.restype = C.c_uint64
        L.orc_n_bonds.argtypes = [C.c_int, C.c_int]
        L.orc_n_bonds.restype = C.c_int64
        L.orc_energy.argtypes = [f32p, C.c_int, C.c_int, C.c_double]
        L.orc_energy.restype = C.c_double
        L.orc_sample_energy.argtypes = [f32p, u8p, C.c_int, C.c_int, C.c_double, C.POINTER(C.c_int64)]
        L.orc_sample_energy.restype = C.c_double
        L.orc_sg_slope.argtypes = [f64p, C.c_int]
        L.orc_sg_slope.restype = C.c_double
        L.orc_equilibrate.argtypes = [f32p, u8p, C.c_int, C.c_int, C.c_double, C.c_double,
                                      C.c_uint64, C.c_uint32, C.c_int, C.c_int, C.c_int, C.c_int,
                                      C.c_double, C.c_double, C.POINTER(C.c_uint32),
                                      C.POINTER(C.c_double), C.POINTER(C.c_double),
                                      C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_equilibrate.restype = C.c_int
        L.orc_simulate.argtypes = [f32p, u8p, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                   C.c_uint64, C.c_uint32, C.c_int, C.c_int, C.c_int,
                                   C.POINTER(C.c_uint32), f64p]
        L.orc_simulate.restype = None
        L.orc_simulate2.argtypes = [f32p, u8p, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                    C.c_uint64, C.c_uint32, C.c_int, C.c_int, C.c_int,
                                    C.POINTER(C.c_uint32), f64p, f64p]
        L.orc_simulate2.restype = None
        L.orc_predict_std.argtypes = [f64p, f64p, C.c_int, u8p, C.c_int64, _CREAL, _CREAL, f32p]
        L.orc_predict_std.restype = None
        L.orc_inv_norm_cdf.argtypes = [C.c_double]
        L.orc_inv_norm_cdf.restype = C.c_double
        L.orc_predict_quantile.argtypes = [f64p, f64p, C.c_int, C.c_double, f32p, u8p, C.c_int64, _CREAL, _CREAL, f32p]
        L.orc_predict_quantile.restype = None
        L.orc_predict.argtypes = [f64p, C.c_int, f32p, u8p, C.c_int64, _CREAL, _CREAL, f32p]
        L.orc_predict.restype = None
        L.orc_num_threads.restype = C.c_int
        L.orc_set_num_threads.argtypes = [C.c_int]
        L.orc_real_bytes.restype = C.c_int
        assert L.orc_real_bytes() == np.dtype(REAL).itemsize
        _lib = L
    return _lib


# ---------------------------------------------------------------------------
# thin functional wrappers (numpy in, numpy out)
# ---------------------------------------------------------------------------
def philox4x32_10(counter, key) -> np.ndarray:
    c = np.ascontiguousarray(counter, dtype=np.uint32)
    k = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.empty(4, dtype=np.uint32)
    lib().orc_philox4x32_10(c, k, out)
    return out


def u01(x: int) -> float:
    return lib().orc_u01(int(x) & 0xFFFFFFFF)


def minmax(z: np.ndarray, mask: np.ndarray):
    zf = np.ascontiguousarray(z, dtype=REAL).ravel()
    m = np.ascontiguousarray(mask, dtype=np.uint8).ravel()
    lo, hi = _CREAL(), _CREAL()
    n = lib().orc_minmax(zf, m, zf.size, C.byref(lo), C.byref(hi))
    return REAL(lo.value), REAL(hi.value), int(n)


def eq1(z, zmin, zmax):
    return REAL(lib().orc_eq1(float(z), float(zmin), float(zmax)))


def transform(z: np.ndarray, mask: np.ndarray, seed: int, g: int = 0):
    """O1 + O2: returns (phi float32 [rows, cols], zmin, zmax)."""
    rows, cols = z.shape
    zf = np.ascontiguousarray(z, dtype=REAL)
    m = np.ascontiguousarray(mask, dtype=np.uint8)
    zmin, zmax, _ = minmax(zf, m)
    phi = np.empty((rows, cols), dtype=REAL)
    lib().orc_transform(zf, m, rows, cols, seed, g, float(zmin), float(zmax), phi)
    return phi, zmin, zmax


def local_energy(phi, Cs, Ss, q) -> float:
    return lib().orc_local_energy(phi, Cs, Ss, q)


def or_reflect(phi, Cs, Ss, q, mode=0, C1=0.0, S1=0.0):
    kept, raw = C.c_int(), C.c_double()
    p = lib().orc_or_reflect(phi, Cs, Ss, C1, S1, q, mode, C.byref(kept), C.byref(raw))
    return p, bool(kept.value), raw.value


def sweep(phi: np.ndarray, mask: np.ndarray, q, T, a, seed, g, t, or_mode=0, diag=False):
    """One UPDATE sweep IN PLACE on phi (float32 [rows, cols]); returns the
    accepted count, plus (margin, edge, R) double arrays when diag=True."""
    rows, cols = phi.shape
    assert phi.dtype == REAL and phi.flags.c_contiguous
    m = np.ascontiguousarray(mask, dtype=np.uint8)
    if diag:
        mg = np.full((rows, cols), np.inf)
        ed = np.full((rows, cols), np.inf)
        RR = np.full((rows, cols), np.inf)
        acc = lib().orc_sweep(phi, m, rows, cols, q, T, a, seed, g, t, or_mode,
                              mg.ctypes.data, ed.ctypes.data, RR.ctypes.data)
        return int(acc), mg, ed, RR
    return int(lib().orc_sweep(phi, m, rows, cols, q, T, a, seed, g, t, or_mode, None, None, None))


def n_bonds(rows, cols) -> int:
    return int(lib().orc_n_bonds(rows, cols))


def energy(phi: np.ndarray, q=0.5) -> float:
    rows, cols = phi.shape
    return lib().orc_energy(np.ascontiguousarray(phi, dtype=REAL), rows, cols, q)


def energy_per_bond(phi: np.ndarray, q=0.5) -> float:
    return energy(phi, q) / n_bonds(*phi.shape)


def sg_slope(e) -> float:
    e = np.ascontiguousarray(e, dtype=np.float64)
    return lib().orc_sg_slope(e, e.size)


@dataclass
class Params:
    """Alg. 2 step 1 parameters; defaults = reading R7."""
    q: float = 0.5
    equil_cap: int = 500
    sweeps_per_real: int = 1
    M: int = 100
    seed: int = 0
    n_f: int = 5
    n_fit: int = 20
    A_targ: float = 0.3
    k_a: float = 3.0
    or_mode: int = 0
    a_eq_mode: int = 0


def equilibrate(phi, mask, T, p: Params, g=0, t0=0, history=False):
    rows, cols = phi.shape
    m = np.ascontiguousarray(mask, dtype=np.uint8)
    t = C.c_uint32(t0)
    a, k = C.c_double(), C.c_double()
    if history:
        eh = np.zeros(p.equil_cap + 2); Ah = np.zeros(p.equil_cap + 2); ah = np.zeros(p.equil_cap + 2)
        ptrs = (eh.ctypes.data, Ah.ctypes.data, ah.ctypes.data)
    else:
        ptrs = (None, None, None)
    i = lib().orc_equilibrate(phi, m, rows, cols, p.q, float(T), p.seed, g, p.or_mode,
                              p.equil_cap, p.n_f, p.n_fit, p.A_targ, p.k_a,
                              C.byref(t), C.byref(a), C.byref(k), *ptrs)
    out = {"sweeps": int(i), "a": a.value, "k": k.value, "t": int(t.value)}
    if history:
        out.update(e_hist=eh[: i + 1], A_hist=Ah[: i + 1], a_hist=ah[: i + 1])
    return out


def simulate(phi, mask, T, a_eq, p: Params, g=0, t0=0):
    rows, cols = phi.shape
    m = np.ascontiguousarray(mask, dtype=np.uint8)
    t = C.c_uint32(t0)
    acc = np.zeros((rows, cols), dtype=np.float64)
    lib().orc_simulate(phi, m, rows, cols, p.q, float(T), float(a_eq), p.seed, g, p.or_mode,
                       p.M, p.sweeps_per_real, C.byref(t), acc.reshape(-1))
    return acc, int(t.value)


def simulate_stats(phi, mask, T, a_eq, p: Params, g=0, t0=0):
    """Step 6 with the sums of phi and of phi^2 over the realizations: (acc, acc2, t)."""
    rows, cols = phi.shape
    m = np.ascontiguousarray(mask, dtype=np.uint8)
    t = C.c_uint32(t0)
    acc = np.zeros((rows, cols), dtype=np.float64)
    acc2 = np.zeros((rows, cols), dtype=np.float64)
    lib().orc_simulate2(phi, m, rows, cols, p.q, float(T), float(a_eq), p.seed, g, p.or_mode,
                        p.M, p.sweeps_per_real, C.byref(t), acc.reshape(-1), acc2.reshape(-1))
    return acc, acc2, int(t.value)


def chains_realizations(M: int, chains: int) -> int:
    """Realizations per chain when M are asked of `chains` chains: ceil(M / chains) (reading R25)."""
    return -(-int(M) // int(chains))


def simulate_chains(phi, mask, T, a_eq, p: Params, chains: int, g=0, batch=1, t0=0):
    """Step 6 run as `chains` independent chains (reading R25; a variant of the paper's single
    chain): every chain starts from the same equilibrated state `phi` (left untouched) at the same sweep index t0,
    chain c draws from the Philox grid word g + c * batch, and each makes ceil(M / chains) realizations of s sweeps.
    The sums of phi and phi^2 are pooled.  Returns (acc, acc2, M_total, t_end, final states [chains][rows][cols])."""
    import dataclasses
    Mc = chains_realizations(p.M, chains)
    pc = dataclasses.replace(p, M=Mc)
    acc = np.zeros(phi.shape, dtype=np.float64)
    acc2 = np.zeros(phi.shape, dtype=np.float64)
    finals = []
    t_end = t0
    for c in range(chains):
        state = phi.copy()
        a1, a2, t_end = simulate_stats(state, mask, T, a_eq, pc, g=g + c * batch, t0=t0)
        acc += a1
        acc2 += a2
        finals.append(state)
    return acc, acc2, chains * Mc, t_end, np.stack(finals)


def predict_std(acc, acc2, M, mask, zmin, zmax) -> np.ndarray:
    """Sample standard deviation of the M back-transformed realizations at the prediction sites (L212)."""
    m = np.ascontiguousarray(mask, dtype=np.uint8)
    out = np.empty(m.shape, dtype=REAL)
    lib().orc_predict_std(np.ascontiguousarray(acc, dtype=np.float64).reshape(-1),
                          np.ascontiguousarray(acc2, dtype=np.float64).reshape(-1), M, m.reshape(-1), m.size,
                          float(zmin), float(zmax), out.reshape(-1))
    return out


def inv_norm_cdf(p: float) -> float:
    return float(lib().orc_inv_norm_cdf(float(p)))


def predict_quantile(acc, acc2, M, p, z, mask, zmin, zmax) -> np.ndarray:
    """Gaussian p-quantile of the conditional distribution from mean and spread of the M realizations (R26)."""
    zf = np.ascontiguousarray(z, dtype=REAL)
    m = np.ascontiguousarray(mask, dtype=np.uint8)
    out = np.empty_like(zf)
    lib().orc_predict_quantile(np.ascontiguousarray(acc, dtype=np.float64).reshape(-1),
                               np.ascontiguousarray(acc2, dtype=np.float64).reshape(-1), M, float(p), zf.reshape(-1),
                               m.reshape(-1), zf.size, float(zmin), float(zmax), out.reshape(-1))
    return out


def predict(acc, M, z, mask, zmin, zmax) -> np.ndarray:
    zf = np.ascontiguousarray(z, dtype=REAL)
    m = np.ascontiguousarray(mask, dtype=np.uint8)
    out = np.empty_like(zf)
    lib().orc_predict(np.ascontiguousarray(acc, dtype=np.float64).reshape(-1), M, zf.reshape(-1),
                      m.reshape(-1), zf.size, float(zmin), float(zmax), out.reshape(-1))
    return out


def run(z, mask, T, p: Params, g=0):
    """Alg. 2 steps 2, 3, 5, 6, 7 for one grid (T is an input: step 4 is not on
    this path).  Returns dict(pred, phi, stats)."""
    phi, zmin, zmax = transform(z, mask, p.seed, g)
    st = equilibrate(phi, mask, T, p, g=g, t0=0)
    a_eq = st["a"] if p.a_eq_mode == 0 else 1.0
    acc, t_end = simulate(phi, mask, T, a_eq, p, g=g, t0=st["t"])
    pred = predict(acc, p.M, z, mask, zmin, zmax)
    st.update(t_end=t_end, a_eq=a_eq, zmin=zmin, zmax=zmax,
              e_final=energy_per_bond(phi, p.q))
    return {"pred": pred, "phi": phi, "stats": st}


# ---------------------------------------------------------------------------
# Alg. 2 step 4: parameter inference
# ---------------------------------------------------------------------------
def sample_energy(phi: np.ndarray, mask: np.ndarray, q=0.5):
    """Step 4.1, Eq. 4: (e_s, N_SP) over the nearest-neighbour pairs of sample sites (reading R1)."""
    rows, cols = phi.shape
    n = C.c_int64()
    e = lib().orc_sample_energy(np.ascontiguousarray(phi, dtype=REAL),
                                np.ascontiguousarray(mask, dtype=np.uint8), rows, cols, float(q), C.byref(n))
    return float(e), int(n.value)


def energy_table(rows: int, cols: int, Ts, p: Params, n_meas: int):
    """e(T_k, L) of Eq. 5 (L105-109): one unconditional chain per ladder temperature T_k (every node free,
    L109 "the values of the spins can be varied at every grid node"), chain k with Philox grid index k.
    Reading R23 (the paper does not describe these runs): the chain starts from the ordered state phi = pi
    (a uniform start freezes vortices in at low T); burn-in is exactly p.equil_cap sweeps of Alg. 2 steps
    5.1-5.2 (sweep, then a = 1 + (i+1)/k_a while A < A_targ) -- the slope criterion of step 5.4 is not used,
    because from the ordered state the energy RISES towards equilibrium and k >= 0 holds at the first check;
    then n_meas further UPDATE sweeps at the a reached, e = H / N_GP after every sweep, averaged."""
    mask = np.zeros((rows, cols), dtype=np.uint8)
    P = rows * cols
    out = []
    for k, T in enumerate(Ts):
        phi = np.full((rows, cols), REAL(np.pi), dtype=REAL)
        a, t = 1.0, 0
        for i in range(p.equil_cap):
            accepted = sweep(phi, mask, p.q, float(T), a, p.seed, k, t, p.or_mode)
            t += 1
            if accepted / P < p.A_targ:
                a = 1.0 + (i + 1) / p.k_a
        acc = 0.0
        for _ in range(n_meas):
            sweep(phi, mask, p.q, float(T), a, p.seed, k, t, p.or_mode)
            t += 1
            acc += energy_per_bond(phi, p.q)
        out.append(acc / n_meas)
    return np.array(out)


def infer_T(e_s: float, Ts, es) -> float:
    """Step 4.2, T = argmin_T |e_s - e(T, L)| (L111) with e(T, L) the piecewise-linear interpolant of the
    ladder (T_k ascending): the first segment that brackets e_s, else the nearer end (reading R24)."""
    Ts = [float(x) for x in Ts]; es = [float(x) for x in es]
    for k in range(len(Ts) - 1):
        lo, hi = es[k], es[k + 1]
        if min(lo, hi) <= e_s <= max(lo, hi) and hi != lo:
            return Ts[k] + (e_s - lo) / (hi - lo) * (Ts[k + 1] - Ts[k])
    k = min(range(len(Ts)), key=lambda i: abs(es[i] - e_s))
    return Ts[k]


def default_ladder(rows: int, cols: int, e_s: float, factors=(0.25, 0.5, 1.0, 2.0, 4.0)):
    """The ladder of step 4.2 when the caller has none: temperatures T_c f_k around the T_c at which the low-temperature
    equipartition energy per bond equals e_s (reading R15): N - 1 harmonic modes carry T / 2 each (k_B = 1), shared by
    N_GP bonds above the ground state e = -1, so 1 + e_s = (N - 1) T_c / (2 N_GP).  Float32 like the temperatures the
    CUDA path takes."""
    N = rows * cols
    T_c = max(2.0 * n_bonds(rows, cols) * (1.0 + e_s) / (N - 1), 1e-12)
    return [float(np.float32(T_c * float(np.float32(f)))) for f in factors]


def infer_T_auto(phi, mask, p: Params, n_meas: int, factors=(0.25, 0.5, 1.0, 2.0, 4.0)):
    """Alg. 2 step 4 for one grid (L97-111, L186-190): 4.1 e_s (Eq. 4), 4.2 the ladder's e(T_k, L) from unconditional
    chains (Eq. 5) and T-hat = argmin |e_s - e(T, L)| (L111).  Returns (T_hat, e_s, ladder, table)."""
    rows, cols = phi.shape
    e_s, n_sp = sample_energy(phi, mask, p.q)
    if n_sp == 0:
        raise ValueError("no pair of neighbouring samples: e_s is undefined")
    Ts = default_ladder(rows, cols, e_s, factors)
    table = energy_table(rows, cols, Ts, p, n_meas)
    return infer_T(e_s, Ts, table), e_s, Ts, table


# ---------------------------------------------------------------------------
# q learned from the data ("In principle, q can be learned from the data"; reading R28)
# ---------------------------------------------------------------------------
def holdout_mask(mask: np.ndarray, fraction: float, seed: int, g: int = 0) -> np.ndarray:
    """The samples withheld for the validation of q: sample site n = row * cols + col is withheld when its uniform of the
    HOLDOUT stream -- Philox counter (n >> 2, 0, 3, g), word n & 3, the uniform of reading R13 -- is below `fraction`.
    Returns a uint8 array: 1 where a sample is withheld."""
    m = np.ascontiguousarray(mask, dtype=np.uint8)
    key = [seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF]
    flat = m.reshape(-1)
    out = np.zeros(flat.size, dtype=np.uint8)
    for block in range((flat.size + 3) // 4):
        if not flat[4 * block: 4 * block + 4].any():
            continue
        x = philox4x32_10([block, 0, 3, g], key)
        for k in range(4):
            n = 4 * block + k
            if n < flat.size and flat[n] and u01(int(x[k])) < fraction:
                out[n] = 1
    return out.reshape(m.shape)


def learn_q(z, mask, p: Params, qs, fraction: float = 0.2, g: int = 0):
    """Reading R28: leave-out validation over the candidates `qs`.  A fraction of the samples is withheld (holdout_mask);
    for every q the method runs on the remaining samples -- Eq. 1 over them, T from their specific energy (Eq. 4 at this
    q) through the equipartition line (the centre of default_ladder), Alg. 2 steps 5-7 with the parameters `p` -- and is
    scored by the root mean square error of its prediction at the withheld samples.  The learned q is the candidate with
    the smallest score (the first of equals).  Returns (q_hat, scores, temperatures)."""
    import dataclasses
    zf = np.ascontiguousarray(z, dtype=REAL)
    held = holdout_mask(mask, fraction, p.seed, g)
    train = (np.asarray(mask, dtype=np.uint8) & (1 - held)).astype(np.uint8)
    if held.sum() == 0 or train.sum() == 0:
        raise ValueError("the withheld or the remaining sample set is empty")
    scores, Ts = [], []
    for q in qs:
        pq = dataclasses.replace(p, q=float(np.float32(q)))
        phi, _, _ = transform(zf, train, p.seed, g)
        e_s, n_sp = sample_energy(phi, train, pq.q)
        if n_sp == 0:
            raise ValueError("no pair of neighbouring samples")
        T = default_ladder(zf.shape[0], zf.shape[1], e_s, (1.0,))[0]
        res = run(zf, train, T, pq, g=g)
        err = (zf.astype(np.float64) - res["pred"].astype(np.float64))[held == 1]
        scores.append(float(np.sqrt(np.mean(err ** 2))))
        Ts.append(T)
    return float(np.float32(qs[int(np.argmin(scores))])), scores, Ts


def num_threads() -> int:
    return int(lib().orc_num_threads())


def set_num_threads(n: int) -> None:
    lib().orc_set_num_threads(int(n))
