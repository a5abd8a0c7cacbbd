"""Thin Python binding of the C-ABI library (include/mpr.h).

Argument marshalling only: every step of the path runs in the CUDA kernels
behind `libmpr_b200.so`.  PyTorch supplies device memory (tensors) and the
stream; nothing here computes.  There is NO CPU fallback: loading fails
loudly if the library has not been built (`python -m paper_1811_01604_b200.build`),
and every call raises `MprError` on a non-zero status.

Function names mirror the C entry points: mpr_create, mpr_set_params,
mpr_equilibrate, mpr_simulate, mpr_predict, ... ; the `Mpr` class bundles a
context with the tensors it must keep alive.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmpr_b200.so")

STATUS_NAMES = {
    0: "MPR_OK", 1: "MPR_ERR_ARG", 2: "MPR_ERR_NO_SAMPLES", 3: "MPR_ERR_NO_FREE",
    4: "MPR_ERR_DEGENERATE_RANGE", 5: "MPR_ERR_NONFINITE", 6: "MPR_ERR_STATE",
    7: "MPR_ERR_WORKSPACE", 8: "MPR_ERR_CUDA", 9: "MPR_ERR_UNSUPPORTED", 10: "MPR_ERR_COMM", 11: "MPR_ERR_TOO_LARGE",
}
NOALLOC_MAX_ROWS = 16384        # MPR_NOALLOC_MAX_ROWS of include/mpr.h

# every symbol include/mpr.h declares
EXPORTS = (
    "mpr_default_params", "mpr_query_workspace", "mpr_create", "mpr_set_params", "mpr_equilibrate",
    "mpr_simulate", "mpr_predict", "mpr_destroy", "mpr_get_angles", "mpr_set_angles",
    "mpr_set_sweep_index", "mpr_sweep", "mpr_energy", "mpr_get_transform", "mpr_get_mask_bits",
    "mpr_get_stats", "mpr_get_launch_count", "mpr_status_string", "mpr_last_cuda_error",
    "mpr_sample_energy", "mpr_create_unconditional", "mpr_measure_energy", "mpr_energy_table",
    "mpr_infer_temperature", "mpr_predict_std", "mpr_query_workspace_chains", "mpr_create_chains",
    "mpr_predict_quantile", "mpr_set_pass_depth", "mpr_get_tiling",
    "mpr_default_ladder", "mpr_infer_temperature_auto", "mpr_set_grid_group",
    "mpr_slab_halo_bytes", "mpr_slab_local_rows", "mpr_query_workspace_slab", "mpr_create_slab",
    "mpr_query_workspace_learn_q", "mpr_learn_q", "mpr_energy_of_angles_noalloc",
    "mpr64_query_workspace", "mpr64_create", "mpr64_set_params", "mpr64_equilibrate", "mpr64_simulate", "mpr64_predict",
    "mpr64_predict_std", "mpr64_destroy", "mpr64_get_angles", "mpr64_set_angles", "mpr64_set_sweep_index", "mpr64_sweep",
    "mpr64_energy", "mpr64_get_transform", "mpr64_get_stats", "mpr64_get_launch_count",
)


class MprError(RuntimeError):
    def __init__(self, status: int, where: str, detail: str = ""):
        self.status = status
        self.name = STATUS_NAMES.get(status, str(status))
        super().__init__(f"{where}: {self.name}" + (f" ({detail})" if detail else ""))


class mpr_params(C.Structure):
    _fields_ = [
        ("struct_size", C.c_uint32), ("q", C.c_float), ("equil_cap", C.c_uint32),
        ("sweeps_per_real", C.c_uint32), ("M", C.c_uint32), ("n_f", C.c_uint32), ("n_fit", C.c_uint32),
        ("A_targ", C.c_float), ("k_a", C.c_float), ("or_mode", C.c_uint32), ("a_eq_mode", C.c_uint32),
        ("seed", C.c_uint64),
    ]


ALLREDUCE_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.POINTER(C.c_double), C.c_int, C.c_int)
EXCHANGE_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p)


class mpr_slab(C.Structure):
    _fields_ = [
        ("struct_size", C.c_uint32), ("rows_global", C.c_int), ("cols", C.c_int), ("row_begin", C.c_int),
        ("row_end", C.c_int), ("allreduce", ALLREDUCE_FN), ("exchange", EXCHANGE_FN), ("user", C.c_void_p),
        ("d_send_up", C.c_void_p), ("d_recv_up", C.c_void_p), ("d_send_down", C.c_void_p), ("d_recv_down", C.c_void_p),
    ]


class mpr_stats(C.Structure):
    _fields_ = [
        ("equil_sweeps", C.c_uint32), ("t", C.c_uint32), ("equilibrated", C.c_uint32),
        ("realizations", C.c_uint32), ("n_free", C.c_uint64), ("n_samples", C.c_uint64),
        ("n_bonds", C.c_uint64), ("a", C.c_double), ("k", C.c_double), ("A_last", C.c_double),
        ("e_last", C.c_double), ("z_min", C.c_float), ("z_max", C.c_float),
    ]


_lib = None


def lib():
    """The loaded C library; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(
                f"{LIB_PATH} is missing: build it with `python -m paper_1811_01604_b200.build` "
                "(the MPR path has no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i, u32, u64, sz = C.c_void_p, C.c_int, C.c_uint32, C.c_uint64, C.c_size_t
        L.mpr_default_params.argtypes = [C.POINTER(mpr_params)]; L.mpr_default_params.restype = None
        L.mpr_query_workspace.argtypes = [i, i, i, C.POINTER(sz)]
        L.mpr_create.argtypes = [C.POINTER(vp), i, i, i, vp, vp, vp, sz, vp]
        L.mpr_query_workspace_chains.argtypes = [i, i, i, i, C.POINTER(sz)]
        L.mpr_create_chains.argtypes = [C.POINTER(vp), i, i, i, i, vp, vp, vp, sz, vp]
        L.mpr_set_params.argtypes = [vp, C.POINTER(mpr_params), C.POINTER(C.c_float)]
        L.mpr_equilibrate.argtypes = [vp]
        L.mpr_simulate.argtypes = [vp]
        L.mpr_predict.argtypes = [vp, vp]
        L.mpr_destroy.argtypes = [vp]
        L.mpr_get_angles.argtypes = [vp, vp]
        L.mpr_set_angles.argtypes = [vp, vp]
        L.mpr_set_sweep_index.argtypes = [vp, u32]
        L.mpr_sweep.argtypes = [vp, u32, C.c_double, C.POINTER(u64)]
        L.mpr_energy.argtypes = [vp, C.POINTER(C.c_double)]
        L.mpr_get_transform.argtypes = [vp, C.POINTER(C.c_float), C.POINTER(C.c_float)]
        L.mpr_get_mask_bits.argtypes = [vp, vp]
        L.mpr_get_stats.argtypes = [vp, C.POINTER(mpr_stats)]
        L.mpr_get_launch_count.argtypes = [vp, C.POINTER(u64)]
        L.mpr_set_pass_depth.argtypes = [vp, u32]
        L.mpr_set_grid_group.argtypes = [vp, i]
        L.mpr_get_tiling.argtypes = [vp, C.POINTER(i), C.POINTER(i), C.POINTER(i), C.POINTER(u32)]
        L.mpr_predict_std.argtypes = [vp, vp]
        L.mpr_predict_quantile.argtypes = [vp, C.c_double, vp]
        L.mpr_sample_energy.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(u64)]
        L.mpr_create_unconditional.argtypes = [C.POINTER(vp), i, i, i, vp, sz, vp]
        L.mpr_measure_energy.argtypes = [vp, u32, C.POINTER(C.c_double)]
        L.mpr_energy_table.argtypes = [i, i, C.POINTER(mpr_params), C.POINTER(C.c_float), i, u32, vp, sz, vp,
                                       C.POINTER(C.c_double)]
        L.mpr_infer_temperature.argtypes = [C.POINTER(C.c_float), C.POINTER(C.c_double), i, C.c_double,
                                            C.POINTER(C.c_double)]
        L.mpr_default_ladder.argtypes = [i, i, C.c_double, C.POINTER(C.c_float), i, C.POINTER(C.c_float)]
        L.mpr_infer_temperature_auto.argtypes = [vp, C.POINTER(mpr_params), C.POINTER(C.c_float), i, u32, vp, sz,
                                                 C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.mpr_slab_halo_bytes.argtypes = [i]
        L.mpr_slab_local_rows.argtypes = [C.POINTER(mpr_slab), C.POINTER(i), C.POINTER(i)]
        L.mpr_query_workspace_slab.argtypes = [C.POINTER(mpr_slab), C.POINTER(sz)]
        L.mpr_create_slab.argtypes = [C.POINTER(vp), C.POINTER(mpr_slab), vp, vp, vp, sz, vp]
        L.mpr_energy_of_angles_noalloc.argtypes = [vp, i, i, C.c_double, vp, vp]
        L.mpr_query_workspace_learn_q.argtypes = [i, i, C.POINTER(sz)]
        L.mpr_learn_q.argtypes = [i, i, vp, vp, C.POINTER(mpr_params), C.POINTER(C.c_float), i, C.c_double, vp, sz, vp,
                                  C.POINTER(C.c_float), C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.mpr64_query_workspace.argtypes = [i, i, C.POINTER(sz)]
        L.mpr64_create.argtypes = [C.POINTER(vp), i, i, vp, vp, vp, sz, vp]
        L.mpr64_set_params.argtypes = [vp, C.POINTER(mpr_params), C.c_double]
        for name in ("mpr64_equilibrate", "mpr64_simulate", "mpr64_destroy"):
            getattr(L, name).argtypes = [vp]
        for name in ("mpr64_predict", "mpr64_predict_std", "mpr64_get_angles", "mpr64_set_angles"):
            getattr(L, name).argtypes = [vp, vp]
        L.mpr64_set_sweep_index.argtypes = [vp, u32]
        L.mpr64_sweep.argtypes = [vp, u32, C.c_double, C.POINTER(u64)]
        L.mpr64_energy.argtypes = [vp, C.POINTER(C.c_double)]
        L.mpr64_get_transform.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.mpr64_get_stats.argtypes = [vp, C.POINTER(mpr_stats)]
        L.mpr64_get_launch_count.argtypes = [vp, C.POINTER(u64)]
        for name in EXPORTS:
            getattr(L, name).restype = C.c_int
        L.mpr_default_params.restype = None
        L.mpr_slab_halo_bytes.restype = C.c_size_t
        L.mpr_status_string.argtypes = [i]; L.mpr_status_string.restype = C.c_char_p
        L.mpr_last_cuda_error.argtypes = []; L.mpr_last_cuda_error.restype = C.c_char_p
        _lib = L
    return _lib


def _check(status: int, where: str):
    if status != 0:
        detail = lib().mpr_last_cuda_error().decode() if status in (8, 11) else lib().mpr_status_string(status).decode()
        raise MprError(status, where, detail)


def default_params(**overrides) -> mpr_params:
    p = mpr_params()
    lib().mpr_default_params(C.byref(p))
    for k, v in overrides.items():
        if not hasattr(p, k):
            raise AttributeError(k)
        setattr(p, k, v)
    return p


def mpr_query_workspace(batch: int, rows: int, cols: int) -> int:
    n = C.c_size_t()
    _check(lib().mpr_query_workspace(batch, rows, cols, C.byref(n)), "mpr_query_workspace")
    return int(n.value)


def mpr_query_workspace_chains(batch: int, chains: int, rows: int, cols: int) -> int:
    n = C.c_size_t()
    _check(lib().mpr_query_workspace_chains(batch, chains, rows, cols, C.byref(n)), "mpr_query_workspace_chains")
    return int(n.value)


@dataclass
class Stats:
    equil_sweeps: int
    t: int
    equilibrated: bool
    realizations: int
    n_free: int
    n_samples: int
    n_bonds: int
    a: float
    k: float
    A_last: float
    e_last: float
    z_min: float
    z_max: float


class Mpr:
    """One context = `batch` grids of rows x cols on one GPU.

    values: float32 CUDA tensor [batch, rows, cols] (or [rows, cols]);
    sample_mask: uint8 CUDA tensor of the same shape, 1 = sample (fixed).
    """

    def __init__(self, values, sample_mask, stream=None, unconditional=None, chains: int = 1):
        import torch
        self.chains = int(chains)
        if unconditional is not None:
            # (batch, rows, cols, device): mpr_create_unconditional, every node free, no data
            self.batch, self.rows, self.cols, self.device = unconditional
            self._torch = torch
            self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            nbytes = mpr_query_workspace(self.batch, self.rows, self.cols)
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self._ctx = C.c_void_p()
            _check(lib().mpr_create_unconditional(C.byref(self._ctx), self.batch, self.rows, self.cols,
                                                  self.workspace.data_ptr(), nbytes, self._stream.cuda_stream),
                   "mpr_create_unconditional")
            self.params = None
            return
        if not values.is_cuda or not sample_mask.is_cuda:
            raise ValueError("values and sample_mask must be CUDA tensors (there is no CPU path)")
        if values.dim() == 2:
            values, sample_mask = values[None], sample_mask[None]
        if values.dtype != torch.float32 or sample_mask.dtype != torch.uint8 or values.shape != sample_mask.shape:
            raise ValueError("values float32 and sample_mask uint8 of the same [batch, rows, cols] shape")
        values, sample_mask = values.contiguous(), sample_mask.contiguous()
        self.device = values.device
        self.batch, self.rows, self.cols = (int(x) for x in values.shape)
        self._torch = torch
        self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        nbytes = mpr_query_workspace_chains(self.batch, self.chains, self.rows, self.cols)
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        assert self.workspace.data_ptr() % 256 == 0
        self._ctx = C.c_void_p()
        if self.chains == 1:
            _check(lib().mpr_create(C.byref(self._ctx), self.batch, self.rows, self.cols,
                                    values.data_ptr(), sample_mask.data_ptr(),
                                    self.workspace.data_ptr(), nbytes, self._stream.cuda_stream), "mpr_create")
        else:
            _check(lib().mpr_create_chains(C.byref(self._ctx), self.batch, self.chains, self.rows, self.cols,
                                           values.data_ptr(), sample_mask.data_ptr(),
                                           self.workspace.data_ptr(), nbytes, self._stream.cuda_stream), "mpr_create_chains")
        self.params = None

    # -- lifecycle ---------------------------------------------------------
    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx.value:
            self._stream.synchronize()
            lib().mpr_destroy(self._ctx)
            self._ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the path ----------------------------------------------------------
    def set_params(self, T, params: mpr_params | None = None, **overrides):
        p = params if params is not None else default_params(**overrides)
        if params is not None:
            for k, v in overrides.items():
                setattr(p, k, v)
        Ts = [float(T)] * self.batch if not hasattr(T, "__len__") else [float(x) for x in T]
        if len(Ts) != self.batch:
            raise ValueError("one temperature per grid")
        arr = (C.c_float * self.batch)(*Ts)
        _check(lib().mpr_set_params(self._ctx, C.byref(p), arr), "mpr_set_params")
        self.params = p
        return self

    def equilibrate(self):
        _check(lib().mpr_equilibrate(self._ctx), "mpr_equilibrate")
        return self

    def simulate(self):
        _check(lib().mpr_simulate(self._ctx), "mpr_simulate")
        return self

    def predict(self, out=None):
        torch = self._torch
        if out is None:
            out = torch.empty((self.batch, self.rows, self.cols), dtype=torch.float32, device=self.device)
        _check(lib().mpr_predict(self._ctx, out.data_ptr()), "mpr_predict")
        return out

    def predict_std(self, out=None):
        torch = self._torch
        if out is None:
            out = torch.empty((self.batch, self.rows, self.cols), dtype=torch.float32, device=self.device)
        _check(lib().mpr_predict_std(self._ctx, out.data_ptr()), "mpr_predict_std")
        return out

    def predict_quantile(self, p: float, out=None):
        torch = self._torch
        if out is None:
            out = torch.empty((self.batch, self.rows, self.cols), dtype=torch.float32, device=self.device)
        _check(lib().mpr_predict_quantile(self._ctx, float(p), out.data_ptr()), "mpr_predict_quantile")
        return out

    # -- Alg. 2 step 4 -------------------------------------------------------
    @classmethod
    def unconditional(cls, batch: int, rows: int, cols: int, device, stream=None):
        return cls(None, None, stream=stream, unconditional=(int(batch), int(rows), int(cols), device))

    def sample_energy(self):
        """(e_s, N_SP) per grid: Eq. 4."""
        e, n = (C.c_double * self.batch)(), (C.c_uint64 * self.batch)()
        _check(lib().mpr_sample_energy(self._ctx, e, n), "mpr_sample_energy")
        return [float(x) for x in e], [int(x) for x in n]

    def measure_energy(self, n_sweeps: int):
        e = (C.c_double * self.batch)()
        _check(lib().mpr_measure_energy(self._ctx, int(n_sweeps), e), "mpr_measure_energy")
        return [float(x) for x in e]

    # -- diagnostics -------------------------------------------------------
    def get_angles(self, out=None):
        torch = self._torch
        if out is None:
            out = torch.empty((self.batch, self.rows, self.cols), dtype=torch.float32, device=self.device)
        _check(lib().mpr_get_angles(self._ctx, out.data_ptr()), "mpr_get_angles")
        return out

    def set_angles(self, phi):
        phi = phi.to(device=self.device, dtype=self._torch.float32).reshape(self.batch, self.rows, self.cols).contiguous()
        _check(lib().mpr_set_angles(self._ctx, phi.data_ptr()), "mpr_set_angles")
        self._stream.synchronize()          # phi may be a temporary
        return self

    def set_sweep_index(self, t: int):
        _check(lib().mpr_set_sweep_index(self._ctx, int(t)), "mpr_set_sweep_index")
        return self

    def sweep(self, n_sweeps: int, a: float, count: bool = False):
        if count:
            acc = (C.c_uint64 * self.batch)()
            _check(lib().mpr_sweep(self._ctx, int(n_sweeps), float(a), acc), "mpr_sweep")
            return [int(x) for x in acc]
        _check(lib().mpr_sweep(self._ctx, int(n_sweeps), float(a), None), "mpr_sweep")
        return None

    def energy(self):
        e = (C.c_double * self.batch)()
        _check(lib().mpr_energy(self._ctx, e), "mpr_energy")
        return [float(x) for x in e]

    def get_transform(self):
        lo, hi = (C.c_float * self.batch)(), (C.c_float * self.batch)()
        _check(lib().mpr_get_transform(self._ctx, lo, hi), "mpr_get_transform")
        return [float(x) for x in lo], [float(x) for x in hi]

    def get_mask_bits(self):
        torch = self._torch
        words = (self.rows * self.cols + 31) // 32
        out = torch.empty((self.batch, words), dtype=torch.int32, device=self.device)
        _check(lib().mpr_get_mask_bits(self._ctx, out.data_ptr()), "mpr_get_mask_bits")
        return out

    def get_stats(self):
        arr = (mpr_stats * self.batch)()
        _check(lib().mpr_get_stats(self._ctx, arr), "mpr_get_stats")
        return [Stats(s.equil_sweeps, s.t, bool(s.equilibrated), s.realizations, s.n_free, s.n_samples,
                      s.n_bonds, s.a, s.k, s.A_last, s.e_last, s.z_min, s.z_max) for s in arr]

    def launch_count(self) -> int:
        n = C.c_uint64()
        _check(lib().mpr_get_launch_count(self._ctx, C.byref(n)), "mpr_get_launch_count")
        return int(n.value)

    def set_pass_depth(self, k: int):
        _check(lib().mpr_set_pass_depth(self._ctx, int(k)), "mpr_set_pass_depth")
        return self

    def set_grid_group(self, grids: int):
        _check(lib().mpr_set_grid_group(self._ctx, int(grids)), "mpr_set_grid_group")
        return self

    def get_tiling(self):
        """(tile rows, tile cols, halo, sweeps per pass)"""
        tr, tc, h, k = C.c_int(), C.c_int(), C.c_int(), C.c_uint32()
        _check(lib().mpr_get_tiling(self._ctx, C.byref(tr), C.byref(tc), C.byref(h), C.byref(k)), "mpr_get_tiling")
        return int(tr.value), int(tc.value), int(h.value), int(k.value)


def slab_local_rows(rows_global: int, cols: int, row_begin: int, row_end: int):
    """mpr_slab_local_rows: (first row, number of rows) of the whole grid a slab holds (own rows plus ghost rows)."""
    sl = mpr_slab(struct_size=C.sizeof(mpr_slab), rows_global=rows_global, cols=cols, row_begin=row_begin, row_end=row_end)
    first, n = C.c_int(), C.c_int()
    _check(lib().mpr_slab_local_rows(C.byref(sl), C.byref(first), C.byref(n)), "mpr_slab_local_rows")
    return int(first.value), int(n.value)


class MprSlab(Mpr):
    """One slab of a grid that is cut into row blocks over several contexts (mpr_create_slab).

    values / sample_mask: CUDA tensors [n_rows, cols] holding the rows slab_local_rows() names (own rows plus ghost rows).
    comm: the transport between the slabs, an object with
        allreduce(values: list[float], op: int) -> list[float]        (op 0 sum, 1 min, 2 max over all slabs)
        exchange(send_up, recv_up, send_down, recv_down, stream)      (uint8 CUDA tensors or None at the grid's edge:
            after it, recv_up holds the upper neighbour's send_down and recv_down the lower neighbour's send_up)
    The other calls are those of Mpr; the outputs have the local shape, `own` is the slice of the own rows in them."""

    def __init__(self, values, sample_mask, rows_global: int, row_begin: int, row_end: int, comm, stream=None):
        import torch
        if values.dim() != 2 or values.dtype != torch.float32 or sample_mask.dtype != torch.uint8 or values.shape != sample_mask.shape:
            raise ValueError("values float32 and sample_mask uint8 of the same [n_rows, cols] shape")
        values, sample_mask = values.contiguous(), sample_mask.contiguous()
        self.chains, self.batch = 1, 1
        self.device = values.device
        self.rows, self.cols = (int(x) for x in values.shape)
        self._torch = torch
        self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        first, n = slab_local_rows(rows_global, self.cols, row_begin, row_end)
        if n != self.rows:
            raise ValueError(f"the slab holds rows [{first}, {first + n}) of the grid: {n} rows, got {self.rows}")
        self.first_row, self.own = first, slice(row_begin - first, row_end - first)
        nbytes = int(lib().mpr_slab_halo_bytes(self.cols))
        up, down = row_begin > 0, row_end < rows_global
        buf = lambda on: torch.zeros(nbytes, dtype=torch.uint8, device=self.device) if on else None
        self._halo = [buf(up), buf(up), buf(down), buf(down)]          # send_up, recv_up, send_down, recv_down
        self.comm = comm
        self.comm_error = None

        def allreduce(_user, vals, n_vals, op):
            try:
                out = comm.allreduce([vals[k] for k in range(n_vals)], int(op))
                for k in range(n_vals):
                    vals[k] = out[k]
                return 0
            except Exception as e:               # an exception must not cross the C frames
                self.comm_error = e
                return 1

        def exchange(_user, _stream):
            try:
                comm.exchange(*self._halo, self._stream)
                return 0
            except Exception as e:
                self.comm_error = e
                return 1

        self._cb = (ALLREDUCE_FN(allreduce), EXCHANGE_FN(exchange))     # kept alive with the context
        ptr = lambda t: t.data_ptr() if t is not None else None
        self._slab = mpr_slab(struct_size=C.sizeof(mpr_slab), rows_global=rows_global, cols=self.cols, row_begin=row_begin,
                              row_end=row_end, allreduce=self._cb[0], exchange=self._cb[1], user=None,
                              d_send_up=ptr(self._halo[0]), d_recv_up=ptr(self._halo[1]),
                              d_send_down=ptr(self._halo[2]), d_recv_down=ptr(self._halo[3]))
        n_ws = C.c_size_t()
        _check(lib().mpr_query_workspace_slab(C.byref(self._slab), C.byref(n_ws)), "mpr_query_workspace_slab")
        self.workspace = torch.empty(int(n_ws.value), dtype=torch.uint8, device=self.device)
        self._ctx = C.c_void_p()
        _check(lib().mpr_create_slab(C.byref(self._ctx), C.byref(self._slab), values.data_ptr(), sample_mask.data_ptr(),
                                     self.workspace.data_ptr(), int(n_ws.value), self._stream.cuda_stream), "mpr_create_slab")
        self.params = None


class DistSlabComm:
    """Transport of MprSlab over torch.distributed: slab r is rank r of `group`, its neighbours ranks r - 1 (up) and r + 1.
    With the nccl backend the halo rows go GPU to GPU (NVLink) by batched send / recv; with gloo they are staged through
    host memory (the CPU tests, or a box without peer access).  Plumbing only."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        self.host = dist.get_backend(group) != "nccl"

    def allreduce(self, values, op):
        import torch
        dist = self.dist
        t = torch.tensor(values, dtype=torch.float64)
        if not self.host:
            t = t.cuda()
        dist.all_reduce(t, op=(dist.ReduceOp.SUM, dist.ReduceOp.MIN, dist.ReduceOp.MAX)[op], group=self.group)
        return [float(x) for x in t.cpu()]

    def exchange(self, send_up, recv_up, send_down, recv_down, stream):
        import torch
        dist = self.dist
        stream.synchronize()                       # the library's copies into the send buffers are done
        ops, staged = [], []
        for send, recv, peer in ((send_up, recv_up, self.rank - 1), (send_down, recv_down, self.rank + 1)):
            if send is None:
                continue
            if self.host:
                s_h, r_h = send.cpu(), torch.empty(recv.shape, dtype=recv.dtype)
                staged.append((recv, r_h))
                send, recv = s_h, r_h
            ops += [dist.P2POp(dist.isend, send, peer, self.group), dist.P2POp(dist.irecv, recv, peer, self.group)]
        for w in (dist.batch_isend_irecv(ops) if ops else []):
            w.wait()
        for dev_t, host_t in staged:
            dev_t.copy_(host_t)
        if not self.host:
            torch.cuda.current_stream().synchronize()


class Mpr64:
    """The double-precision path (mpr64_* calls): one grid of rows x cols.

    values: float64 CUDA tensor [rows, cols]; sample_mask: uint8 CUDA tensor of the same shape, 1 = sample (fixed).
    """

    def __init__(self, values, sample_mask, stream=None):
        import torch
        if not values.is_cuda or not sample_mask.is_cuda:
            raise ValueError("values and sample_mask must be CUDA tensors (there is no CPU path)")
        if values.dtype != torch.float64 or sample_mask.dtype != torch.uint8 or values.shape != sample_mask.shape or values.dim() != 2:
            raise ValueError("values float64 and sample_mask uint8 of the same [rows, cols] shape")
        values, sample_mask = values.contiguous(), sample_mask.contiguous()
        self.device = values.device
        self.rows, self.cols = (int(x) for x in values.shape)
        self._torch = torch
        self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        n = C.c_size_t()
        _check(lib().mpr64_query_workspace(self.rows, self.cols, C.byref(n)), "mpr64_query_workspace")
        self.workspace = torch.empty(int(n.value), dtype=torch.uint8, device=self.device)
        self._ctx = C.c_void_p()
        _check(lib().mpr64_create(C.byref(self._ctx), self.rows, self.cols, values.data_ptr(), sample_mask.data_ptr(),
                                  self.workspace.data_ptr(), int(n.value), self._stream.cuda_stream), "mpr64_create")
        self.params = None

    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx.value:
            self._stream.synchronize()
            lib().mpr64_destroy(self._ctx)
            self._ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_params(self, T, params: mpr_params | None = None, **overrides):
        p = params if params is not None else default_params(**overrides)
        if params is not None:
            for k, v in overrides.items():
                setattr(p, k, v)
        _check(lib().mpr64_set_params(self._ctx, C.byref(p), float(T)), "mpr64_set_params")
        self.params = p
        return self

    def equilibrate(self):
        _check(lib().mpr64_equilibrate(self._ctx), "mpr64_equilibrate")
        return self

    def simulate(self):
        _check(lib().mpr64_simulate(self._ctx), "mpr64_simulate")
        return self

    def _out(self, out):
        return out if out is not None else self._torch.empty((self.rows, self.cols), dtype=self._torch.float64, device=self.device)

    def predict(self, out=None):
        out = self._out(out)
        _check(lib().mpr64_predict(self._ctx, out.data_ptr()), "mpr64_predict")
        return out

    def predict_std(self, out=None):
        out = self._out(out)
        _check(lib().mpr64_predict_std(self._ctx, out.data_ptr()), "mpr64_predict_std")
        return out

    def get_angles(self, out=None):
        out = self._out(out)
        _check(lib().mpr64_get_angles(self._ctx, out.data_ptr()), "mpr64_get_angles")
        return out

    def set_angles(self, phi):
        phi = phi.to(device=self.device, dtype=self._torch.float64).reshape(self.rows, self.cols).contiguous()
        _check(lib().mpr64_set_angles(self._ctx, phi.data_ptr()), "mpr64_set_angles")
        self._stream.synchronize()          # phi may be a temporary
        return self

    def set_sweep_index(self, t: int):
        _check(lib().mpr64_set_sweep_index(self._ctx, int(t)), "mpr64_set_sweep_index")
        return self

    def sweep(self, n_sweeps: int, a: float, count: bool = False):
        if count:
            acc = C.c_uint64()
            _check(lib().mpr64_sweep(self._ctx, int(n_sweeps), float(a), C.byref(acc)), "mpr64_sweep")
            return int(acc.value)
        _check(lib().mpr64_sweep(self._ctx, int(n_sweeps), float(a), None), "mpr64_sweep")
        return None

    def energy(self) -> float:
        e = C.c_double()
        _check(lib().mpr64_energy(self._ctx, C.byref(e)), "mpr64_energy")
        return float(e.value)

    def get_transform(self):
        lo, hi = C.c_double(), C.c_double()
        _check(lib().mpr64_get_transform(self._ctx, C.byref(lo), C.byref(hi)), "mpr64_get_transform")
        return float(lo.value), float(hi.value)

    def get_stats(self) -> Stats:
        s = mpr_stats()
        _check(lib().mpr64_get_stats(self._ctx, C.byref(s)), "mpr64_get_stats")
        return Stats(s.equil_sweeps, s.t, bool(s.equilibrated), s.realizations, s.n_free, s.n_samples,
                     s.n_bonds, s.a, s.k, s.A_last, s.e_last, s.z_min, s.z_max)

    def launch_count(self) -> int:
        n = C.c_uint64()
        _check(lib().mpr64_get_launch_count(self._ctx, C.byref(n)), "mpr64_get_launch_count")
        return int(n.value)


def energy_table(rows: int, cols: int, Ts, n_meas: int, device, params: mpr_params | None = None, **overrides):
    """mpr_energy_table: e(T_k, L) of Eq. 5 for the ladder Ts from unconditional chains.  Returns a list."""
    import torch
    p = params if params is not None else default_params(**overrides)
    n_T = len(Ts)
    nbytes = mpr_query_workspace(n_T, rows, cols)
    ws = torch.empty(nbytes, dtype=torch.uint8, device=device)
    arr = (C.c_float * n_T)(*[float(x) for x in Ts])
    e = (C.c_double * n_T)()
    stream = torch.cuda.current_stream(device)
    _check(lib().mpr_energy_table(int(rows), int(cols), C.byref(p), arr, n_T, int(n_meas), ws.data_ptr(), nbytes,
                                  stream.cuda_stream, e), "mpr_energy_table")
    return [float(x) for x in e]


def infer_temperature(Ts, es, e_s: float) -> float:
    """mpr_infer_temperature: the ladder's interpolant inverted at e_s."""
    n = len(Ts)
    out = C.c_double()
    _check(lib().mpr_infer_temperature((C.c_float * n)(*[float(x) for x in Ts]), (C.c_double * n)(*[float(x) for x in es]),
                                       n, float(e_s), C.byref(out)), "mpr_infer_temperature")
    return float(out.value)


def default_ladder(rows: int, cols: int, e_s: float, factors=None):
    """mpr_default_ladder: the temperatures step 4.2 uses when the caller has no ladder."""
    n = 5 if factors is None else len(factors)
    f = None if factors is None else (C.c_float * n)(*[float(x) for x in factors])
    out = (C.c_float * n)()
    _check(lib().mpr_default_ladder(int(rows), int(cols), float(e_s), f, n, out), "mpr_default_ladder")
    return [float(x) for x in out]


def infer_T(ctx: "Mpr", n_meas: int = 100, ladder=None, return_e_s: bool = False, **params):
    """mpr_infer_temperature_auto: Alg. 2 step 4 for every grid of a context, in the library (e_s, ladder around the
    equipartition estimate, e(T, L) of the ladder from unconditional chains, inversion).  `ladder` = the factors of
    the ladder (None: the library's).  Returns the list of T-hat (and the list of e_s)."""
    import torch
    p = default_params(**params)
    n_T = 5 if ladder is None else len(ladder)
    f = None if ladder is None else (C.c_float * n_T)(*[float(x) for x in ladder])
    nbytes = mpr_query_workspace(n_T, ctx.rows, ctx.cols)
    ws = torch.empty(nbytes, dtype=torch.uint8, device=ctx.device)
    T_hat, e_s = (C.c_double * ctx.batch)(), (C.c_double * ctx.batch)()
    _check(lib().mpr_infer_temperature_auto(ctx._ctx, C.byref(p), f, n_T, int(n_meas), ws.data_ptr(), nbytes, T_hat, e_s),
           "mpr_infer_temperature_auto")
    if return_e_s:
        return [float(x) for x in T_hat], [float(x) for x in e_s]
    return [float(x) for x in T_hat]


def energy_of_angles_noalloc(phi, q: float = 0.5, out=None, rows: int | None = None, cols: int | None = None):
    """mpr_energy_of_angles_noalloc: energy per bond of the angle field `phi` (float32 CUDA tensor [rows, cols]) into
    `out` (float64 CUDA tensor of one element, made here when None: the CALLER's allocation; the library makes none).
    Asynchronous on the current stream.  `rows` / `cols` override the tensor's shape (tests of the size check)."""
    import torch
    if not phi.is_cuda or phi.dtype != torch.float32 or phi.dim() != 2 or not phi.is_contiguous():
        raise ValueError("phi: a contiguous float32 CUDA tensor [rows, cols]")
    if out is None:
        out = torch.empty(1, dtype=torch.float64, device=phi.device)
    r, c = (int(x) for x in phi.shape)
    stream = torch.cuda.current_stream(phi.device)
    _check(lib().mpr_energy_of_angles_noalloc(phi.data_ptr(), r if rows is None else int(rows), c if cols is None else int(cols),
                                              float(q), out.data_ptr(), stream.cuda_stream), "mpr_energy_of_angles_noalloc")
    return out


def learn_q(values, sample_mask, qs, holdout_fraction: float = 0.2, params: mpr_params | None = None, **overrides):
    """mpr_learn_q: q by leave-out validation over the candidates `qs` on one grid (reading R28).
    Returns (q_hat, scores, temperatures)."""
    import torch
    p = params if params is not None else default_params(**overrides)
    values, sample_mask = values.contiguous(), sample_mask.contiguous()
    rows, cols = (int(x) for x in values.shape[-2:])
    n = C.c_size_t()
    _check(lib().mpr_query_workspace_learn_q(rows, cols, C.byref(n)), "mpr_query_workspace_learn_q")
    ws = torch.empty(int(n.value), dtype=torch.uint8, device=values.device)
    n_q = len(qs)
    q_hat, scores, Ts = C.c_float(), (C.c_double * n_q)(), (C.c_double * n_q)()
    stream = torch.cuda.current_stream(values.device)
    _check(lib().mpr_learn_q(rows, cols, values.data_ptr(), sample_mask.data_ptr(), C.byref(p),
                             (C.c_float * n_q)(*[float(x) for x in qs]), n_q, float(holdout_fraction), ws.data_ptr(),
                             int(n.value), stream.cuda_stream, C.byref(q_hat), scores, Ts), "mpr_learn_q")
    return float(q_hat.value), [float(x) for x in scores], [float(x) for x in Ts]


def interpolate(values, sample_mask, T=None, chains: int = 1, **params):
    """The whole path for a batch of grids: create, (T = None: infer the temperatures, Alg. 2 step 4,) set_params,
    equilibrate, simulate, predict.  Returns (prediction tensor, list of Stats)."""
    m = Mpr(values, sample_mask, chains=chains)
    try:
        if T is None:
            T = infer_T(m, **{k: v for k, v in params.items() if k in ("seed", "q", "equil_cap", "or_mode")})
        m.set_params(T, **params).equilibrate().simulate()
        out = m.predict()
        stats = m.get_stats()
    finally:
        m.close()
    return out, stats
