"""Thin ctypes binding of include/tnmc.h: argument marshalling only.

Same names as the C ABI.  torch is used for device memory and the current stream; every step of
the hot path runs inside libtnmc.so.  Importing this module fails loudly if the library is
missing and cannot be built -- there is no CPU fallback.
"""
import ctypes as C
import os

import torch

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtnmc.so")

TNMC_OK, TNMC_EINVAL, TNMC_ENOMEM, TNMC_ECUDA, TNMC_ESTATE, TNMC_ENUMERIC = range(6)
TNMC_F64, TNMC_F32_LOGSCALE, TNMC_F32_STORE, TNMC_TF32_FAST = 0, 1, 2, 3
FLAG_NAMES = ("rho_zero", "nonfinite", "logz_nonpos", "near_threshold", "jacobi_limit", "sigma_zero",
              "reserved6", "reserved7")
N_FLAGS = 8


def _load():
    if not os.path.exists(LIB_PATH) or _build.needs_build():
        _build.build()
    lib = C.CDLL(LIB_PATH)
    vp, i32, u64, sz, dbl = C.c_void_p, C.c_int, C.c_uint64, C.c_size_t, C.c_double
    lib.tnmc_workspace_bytes.restype = sz
    lib.tnmc_workspace_bytes.argtypes = [i32, i32, i32, i32, i32, i32]
    lib.tnmc_create.restype = i32
    lib.tnmc_create.argtypes = [C.POINTER(vp), i32, i32, dbl, i32, vp, vp, u64, i32, i32, i32, vp, sz, vp]
    lib.tnmc_build_envs.restype = i32
    lib.tnmc_build_envs.argtypes = [vp, vp]
    lib.tnmc_sample.restype = i32
    lib.tnmc_sample.argtypes = [vp, i32, i32, i32, u64, u64, vp, vp]
    lib.tnmc_sample_ex.restype = i32
    lib.tnmc_sample_ex.argtypes = [vp, i32, i32, i32, u64, u64, vp, vp, vp, vp]
    lib.tnmc_sample_fused.restype = i32
    lib.tnmc_sample_fused.argtypes = [vp, i32, i32, i32, u64, u64, vp, vp, vp, vp]
    lib.tnmc_energy.restype = i32
    lib.tnmc_energy.argtypes = [vp, i32, i32, i32, vp, vp]
    lib.tnmc_metropolis.restype = i32
    lib.tnmc_metropolis.argtypes = [vp, i32, i32, i32, vp, vp, u64, u64, vp, vp, vp, vp, vp, vp]
    lib.tnmc_workspace_bytes_real.restype = sz
    lib.tnmc_workspace_bytes_real.argtypes = [i32, i32, i32, i32, i32, i32]
    lib.tnmc_create_real.restype = i32
    lib.tnmc_create_real.argtypes = [C.POINTER(vp), i32, i32, dbl, i32, vp, vp, u64, i32, i32, i32, vp, sz, vp]
    lib.tnmc_energy_real.restype = i32
    lib.tnmc_energy_real.argtypes = [vp, i32, i32, i32, vp, vp]
    lib.tnmc_metropolis_real.restype = i32
    lib.tnmc_metropolis_real.argtypes = [vp, i32, i32, i32, vp, vp, u64, u64, vp, vp, vp, vp, vp, vp]
    lib.tnmc_observables.restype = i32
    lib.tnmc_observables.argtypes = [vp, i32, i32, i32, vp, vp, vp, vp, vp, vp, vp]
    lib.tnmc_observables_real.restype = i32
    lib.tnmc_observables_real.argtypes = [vp, i32, i32, i32, vp, vp, vp, vp, vp, vp, vp]
    lib.tnmc_replica_overlap.restype = i32
    lib.tnmc_replica_overlap.argtypes = [vp, i32, i32, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.tnmc_observables_static_max.restype = sz
    lib.tnmc_observables_static_max.argtypes = []
    lib.tnmc_observables_static.restype = i32
    lib.tnmc_observables_static.argtypes = [vp, i32, i32, i32, vp, vp, vp, vp, vp, vp]
    lib.tnmc_run_host_workspace_bytes.restype = sz
    lib.tnmc_run_host_workspace_bytes.argtypes = [i32, i32, i32, i32, i32, i32]
    lib.tnmc_run_host.restype = i32
    lib.tnmc_run_host.argtypes = [i32, i32, dbl, i32, i32, vp, vp, u64, u64, i32, i32, vp, sz, vp,
                                  vp, vp, vp, vp, vp, vp]
    lib.tnmc_get_flags.restype = i32
    lib.tnmc_get_flags.argtypes = [vp, vp]
    lib.tnmc_get_env_row.restype = i32
    lib.tnmc_get_env_row.argtypes = [vp, i32, i32, vp, vp]
    lib.tnmc_fp64_peak_tflops.restype = dbl
    lib.tnmc_fp64_peak_tflops.argtypes = [i32, vp, vp]
    lib.tnmc_launch_count.restype = u64
    lib.tnmc_launch_count.argtypes = [vp]
    lib.tnmc_last_error.restype = C.c_char_p
    lib.tnmc_last_error.argtypes = [vp]
    lib.tnmc_destroy.restype = None
    lib.tnmc_destroy.argtypes = [vp]
    return lib


lib = _load()


class TnmcError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"tnmc status {status}: {msg}")
        self.status = status


def _check(st, ctx=None):
    if st != TNMC_OK:
        raise TnmcError(st, lib.tnmc_last_error(ctx).decode())


def _ptr(t, dtype=None, device_type="cuda"):
    if t is None:
        return None
    assert t.is_contiguous(), "tensor must be contiguous"
    assert t.device.type == device_type, f"tensor must live on {device_type}"
    if dtype is not None:
        assert t.dtype == dtype, f"expected {dtype}, got {t.dtype}"
    return C.c_void_p(t.data_ptr())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def words(L):
    return (L + 31) // 32


def tnmc_workspace_bytes(L, chi, n_dis, n_samples_max, prec=TNMC_F64, ckpt_stride=0):
    return int(lib.tnmc_workspace_bytes(L, chi, n_dis, n_samples_max, prec, ckpt_stride))


class Context:
    """Owns the torch-allocated workspace and the tnmc_ctx handle (tnmc_create / tnmc_destroy)."""

    def __init__(self, L, chi, beta, Jr, Jd, n_samples_max, first_disorder=0, prec=TNMC_F64,
                 ckpt_stride=0, workspace=None):
        n_dis = Jr.shape[0]
        assert Jr.shape == (n_dis, L, L) and Jd.shape == (n_dis, L, L)
        self.real_j = Jr.dtype == torch.float64           # real-valued couplings -> tnmc_create_real
        wsb = lib.tnmc_workspace_bytes_real if self.real_j else lib.tnmc_workspace_bytes
        need = int(wsb(L, chi, n_dis, n_samples_max, prec, ckpt_stride))
        if need == 0:
            raise TnmcError(TNMC_EINVAL, "tnmc_workspace_bytes: invalid sizes")
        if workspace is None:
            workspace = torch.empty(need, dtype=torch.uint8, device=Jr.device)
        self.workspace = workspace
        self.L, self.chi, self.beta, self.n_dis, self.n_samples_max = L, chi, float(beta), n_dis, n_samples_max
        self.W = words(L)
        self.device = Jr.device
        self._Jr, self._Jd = Jr, Jd          # kept alive until the pack kernel / copy has certainly run
        h = C.c_void_p()
        jt = torch.float64 if self.real_j else torch.int8
        create = lib.tnmc_create_real if self.real_j else lib.tnmc_create
        st = create(C.byref(h), L, chi, float(beta), n_dis, _ptr(Jr, jt), _ptr(Jd, jt),
                    first_disorder, n_samples_max, prec, ckpt_stride,
                    _ptr(workspace, torch.uint8), workspace.numel(), _stream())
        _check(st)
        self.h = h

    def close(self):
        if getattr(self, "h", None) and lib is not None:   # `lib` is None during interpreter shutdown
            lib.tnmc_destroy(self.h)
        self.h = None

    def __del__(self):
        self.close()

    # -- the five entry points ------------------------------------------------------------------
    def tnmc_build_envs(self, logZ=None):
        if logZ is None:
            logZ = torch.empty(self.n_dis, dtype=torch.float64, device=self.device)
        _check(lib.tnmc_build_envs(self.h, _ptr(logZ, torch.float64)), self.h)
        return logZ

    def tnmc_sample(self, n_samples, seed, sample_offset=0, dis_begin=0, dis_count=None, cfg_bits=None,
                    logq=None, forced_cfg_bits=None, probs=None):
        dis_count = self.n_dis - dis_begin if dis_count is None else dis_count
        if cfg_bits is None:
            cfg_bits = torch.empty((dis_count, n_samples, self.L, self.W), dtype=torch.int32, device=self.device)
        if logq is None:
            logq = torch.empty((dis_count, n_samples), dtype=torch.float64, device=self.device)
        if forced_cfg_bits is None and probs is None:
            st = lib.tnmc_sample(self.h, dis_begin, dis_count, n_samples, seed, sample_offset,
                                 _ptr(cfg_bits, torch.int32), _ptr(logq, torch.float64))
        else:
            st = lib.tnmc_sample_ex(self.h, dis_begin, dis_count, n_samples, seed, sample_offset,
                                    _ptr(forced_cfg_bits, torch.int32), _ptr(cfg_bits, torch.int32),
                                    _ptr(logq, torch.float64), _ptr(probs, torch.float64))
        _check(st, self.h)
        return cfg_bits, logq

    def tnmc_sample_fused(self, n_samples, seed, sample_offset=0, dis_begin=0, dis_count=None, keep_cfg=True,
                          cfg_bits=None, logq=None, E=None, M=None):
        """returns (cfg_bits or None, logq, E, M): E and M come out of the sampling sweep itself"""
        dis_count = self.n_dis - dis_begin if dis_count is None else dis_count
        dev = self.device
        if cfg_bits is None and keep_cfg:
            cfg_bits = torch.empty((dis_count, n_samples, self.L, self.W), dtype=torch.int32, device=dev)
        if logq is None:
            logq = torch.empty((dis_count, n_samples), dtype=torch.float64, device=dev)
        if E is None:
            E = torch.empty((dis_count, n_samples), dtype=torch.int32, device=dev)
        if M is None:
            M = torch.empty((dis_count, n_samples), dtype=torch.int32, device=dev)
        _check(lib.tnmc_sample_fused(self.h, dis_begin, dis_count, n_samples, seed, sample_offset,
                                     _ptr(cfg_bits, torch.int32), _ptr(logq, torch.float64),
                                     _ptr(E, torch.int32), _ptr(M, torch.int32)), self.h)
        return cfg_bits, logq, E, M

    def tnmc_energy(self, cfg_bits, dis_begin=0, E=None):
        dis_count, n_samples = cfg_bits.shape[0], cfg_bits.shape[1]
        et = torch.float64 if self.real_j else torch.int32
        if E is None:
            E = torch.empty((dis_count, n_samples), dtype=et, device=self.device)
        fn = lib.tnmc_energy_real if self.real_j else lib.tnmc_energy
        _check(fn(self.h, dis_begin, dis_count, n_samples, _ptr(cfg_bits, torch.int32), _ptr(E, et)), self.h)
        return E

    def tnmc_metropolis(self, E, logq, seed, step_offset=0, dis_begin=0, state=None, want_sum_min1=False):
        dis_count, n_samples = E.shape
        dev = self.device
        if state is None:
            state = (torch.zeros(dis_count, dtype=torch.float64, device=dev),
                     torch.zeros(dis_count, dtype=E.dtype, device=dev),
                     torch.full((dis_count,), -1, dtype=torch.int64, device=dev))
        cur_logq, cur_E, cur_idx = state
        accepted = torch.empty((dis_count, n_samples), dtype=torch.uint8, device=dev)
        n_acc = torch.empty(dis_count, dtype=torch.int64, device=dev)
        smin = torch.empty(dis_count, dtype=torch.float64, device=dev) if want_sum_min1 else None
        et = torch.float64 if self.real_j else torch.int32
        fn = lib.tnmc_metropolis_real if self.real_j else lib.tnmc_metropolis
        _check(fn(self.h, dis_begin, dis_count, n_samples, _ptr(E, et),
                                   _ptr(logq, torch.float64), seed, step_offset,
                                   _ptr(cur_logq, torch.float64), _ptr(cur_E, et),
                                   _ptr(cur_idx, torch.int64), _ptr(accepted, torch.uint8),
                                   _ptr(n_acc, torch.int64), _ptr(smin, torch.float64)), self.h)
        return accepted, n_acc, state, smin

    def tnmc_observables(self, cfg_bits, E, accepted, dis_begin=0, state=None, sums=None):
        """returns (M, (cur_E, cur_M), sums) -- sums (dis_count, 5) accumulates E, E^2, M, |M|, M^2 over the steps"""
        dis_count, n_samples = E.shape
        dev = self.device
        if state is None:
            state = (torch.zeros(dis_count, dtype=E.dtype, device=dev), torch.zeros(dis_count, dtype=torch.int32, device=dev))
        if sums is None:
            sums = torch.zeros((dis_count, 5), dtype=torch.float64, device=dev)
        M = torch.empty((dis_count, n_samples), dtype=torch.int32, device=dev)
        et = torch.float64 if self.real_j else torch.int32
        fn = lib.tnmc_observables_real if self.real_j else lib.tnmc_observables
        _check(fn(self.h, dis_begin, dis_count, n_samples, _ptr(cfg_bits, torch.int32), _ptr(E, et),
                                    _ptr(accepted, torch.uint8), _ptr(M, torch.int32), _ptr(state[0], et),
                                    _ptr(state[1], torch.int32), _ptr(sums, torch.float64)), self.h)
        return M, state, sums

    def tnmc_replica_overlap(self, cfg_a, accepted_a, cfg_b, accepted_b, state=None, sums=None):
        """returns (q_steps, (cur_cfg_a, cur_cfg_b), sums) -- sums (dis_count, 3) accumulates q, |q|, q^2 over the steps"""
        dis_count, n_samples = accepted_a.shape
        dev = self.device
        if state is None:
            state = (torch.zeros((dis_count, self.L, self.W), dtype=torch.int32, device=dev),
                     torch.zeros((dis_count, self.L, self.W), dtype=torch.int32, device=dev))
        if sums is None:
            sums = torch.zeros((dis_count, 3), dtype=torch.float64, device=dev)
        q = torch.empty((dis_count, n_samples), dtype=torch.int32, device=dev)
        _check(lib.tnmc_replica_overlap(self.h, dis_count, n_samples, _ptr(cfg_a, torch.int32), _ptr(accepted_a, torch.uint8),
                                        _ptr(cfg_b, torch.int32), _ptr(accepted_b, torch.uint8), _ptr(state[0], torch.int32),
                                        _ptr(state[1], torch.int32), _ptr(q, torch.int32), _ptr(sums, torch.float64)), self.h)
        return q, state, sums

    def tnmc_observables_static(self, cfg_bits, E, accepted, state, sums, dis_begin=0):
        """tnmc_observables without any allocation: `state` = (cur_E, cur_M) and `sums` are caller tensors, the
        magnetisation scratch is the library's static device array (limit tnmc_observables_static_max proposals)."""
        dis_count, n_samples = E.shape
        _check(lib.tnmc_observables_static(self.h, dis_begin, dis_count, n_samples, _ptr(cfg_bits, torch.int32),
                                           _ptr(E, torch.int32), _ptr(accepted, torch.uint8), _ptr(state[0], torch.int32),
                                           _ptr(state[1], torch.int32), _ptr(sums, torch.float64)), self.h)
        return state, sums

    # -- inspection -----------------------------------------------------------------------------
    def tnmc_get_flags(self):
        out = (C.c_uint64 * N_FLAGS)()
        _check(lib.tnmc_get_flags(self.h, out), self.h)
        return dict(zip(FLAG_NAMES, [int(v) for v in out]))

    def tnmc_get_env_row(self, disorder, row):
        out = torch.empty((self.L, self.chi, 2, self.chi), dtype=torch.float64)
        ls = C.c_double()
        _check(lib.tnmc_get_env_row(self.h, disorder, row, C.c_void_p(out.data_ptr()), C.byref(ls)), self.h)
        return out, ls.value

    def tnmc_launch_count(self):
        return int(lib.tnmc_launch_count(self.h))


def tnmc_run_host_workspace_bytes(L, chi, n_dis, n_samples, prec=TNMC_F64, ckpt_stride=0):
    return int(lib.tnmc_run_host_workspace_bytes(L, chi, n_dis, n_samples, prec, ckpt_stride))


def tnmc_run_host(L, chi, beta, Jr_host, Jd_host, n_samples, seed, workspace, first_disorder=0,
                  prec=TNMC_F64, ckpt_stride=0, out=None, want_cfg=True):
    """Host buffers in, host buffers out (pinned torch CPU tensors); `workspace` is a CUDA uint8 tensor."""
    n_dis = Jr_host.shape[0]
    W = words(L)
    if out is None:
        pin = torch.cuda.is_available()
        out = dict(
            cfg_bits=torch.empty((n_dis, n_samples, L, W), dtype=torch.int32, pin_memory=pin) if want_cfg else None,
            E=torch.empty((n_dis, n_samples), dtype=torch.int32, pin_memory=pin),
            logq=torch.empty((n_dis, n_samples), dtype=torch.float64, pin_memory=pin),
            accepted=torch.empty((n_dis, n_samples), dtype=torch.uint8, pin_memory=pin),
            logZ=torch.empty(n_dis, dtype=torch.float64, pin_memory=pin),
            n_accepted=torch.empty(n_dis, dtype=torch.int64, pin_memory=pin))
    hp = lambda t, dt: _ptr(t, dt, "cpu")
    st = lib.tnmc_run_host(L, chi, float(beta), n_dis, n_samples, hp(Jr_host, torch.int8), hp(Jd_host, torch.int8),
                           first_disorder, seed, prec, ckpt_stride, _ptr(workspace, torch.uint8),
                           workspace.numel(), _stream(), hp(out["cfg_bits"], torch.int32), hp(out["E"], torch.int32),
                           hp(out["logq"], torch.float64), hp(out["accepted"], torch.uint8),
                           hp(out["logZ"], torch.float64), hp(out["n_accepted"], torch.int64))
    _check(st)
    return out


def tnmc_fp64_peak_tflops(which, scratch=None):
    """Live FP64 roofline probe: which=0 scalar DFMA, which=1 DMMA (mma.sync.m8n8k4.f64)."""
    if scratch is None:
        scratch = torch.empty(1 << 20, dtype=torch.uint8, device="cuda")
    v = float(lib.tnmc_fp64_peak_tflops(which, _ptr(scratch, torch.uint8), _stream()))
    if v <= 0:
        raise TnmcError(TNMC_ECUDA, "tnmc_fp64_peak_tflops failed")
    return v
