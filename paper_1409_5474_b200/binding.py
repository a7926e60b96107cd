"""ctypes binding of libnb.so (include/nb.h): same names, argument marshalling only.

torch supplies device memory (`tensor.data_ptr()`) and the stream; every step of the path runs in
the library's sm_100a kernels.  There is no fallback: importing this module without a built
libnb.so raises, and `nb_create` fails on anything that is not a compute-capability-10.x GPU.
"""
import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("NB_LIBRARY") or os.path.join(_HERE, "libnb.so")   # NB_LIBRARY: another build

NB_OK, NB_ERR_ARG, NB_ERR_ALLOC, NB_ERR_CUDA = 0, -1, -2, -3
NB_ERR_INDEX, NB_ERR_STATE, NB_ERR_ARCH, NB_ERR_PEER = -4, -5, -6, -7
NB_XCHG_HANDLE_BYTES = 64
NB_MAX_FLAGGED = 1024
NB_STATIC_NI_MAX = 4096
NB_STATIC_SCRATCH_BYTES = 4194304

EXPORTS = [
    "nb_create", "nb_destroy", "nb_set_stream", "nb_workspace_bytes", "nb_set_workspace",
    "nb_set_j", "nb_update_j", "nb_update_j_host", "nb_set_j_host", "nb_clear", "nb_count", "nb_set_flags",
    "nb_predict", "nb_get_predicted", "nb_force", "nb_force_ext", "nb_force_ext_ids", "nb_force_fused", "nb_set_fused", "nb_force_host", "nb_set_order", "nb_force6", "nb_set_precision", "nb_set_tuning",
    "nb_last_launch", "nb_launch_count", "nb_set_profiling", "nb_kernel_times", "nb_sync",
    "nb_set_dt", "nb_get_state", "nb_init_steps", "nb_next_block", "nb_correct", "nb_step", "nb_steps", "nb_set_steps_bound", "nb_set_steps_queue", "nb_block_forces", "nb_strerror", "nb_version",
    "nb_xchg_create", "nb_xchg_export", "nb_xchg_attach", "nb_xchg_destroy", "nb_xchg_set_timeout", "nb_xforce",
    "nb_force_static",
]

if not os.path.exists(LIB_PATH):
    raise ImportError(
        "paper_1409_5474_b200/libnb.so is missing: build it with "
        "`python -c 'import __graft_entry__ as g; g.build()'` (needs nvcc). There is no fallback.")

lib = ctypes.CDLL(LIB_PATH)

_vp, _i64, _i32, _dbl = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_double
lib.nb_create.argtypes = [ctypes.POINTER(_vp), _i64, _i64, _i32, _vp]
lib.nb_destroy.argtypes = [_vp]
lib.nb_set_stream.argtypes = [_vp, _vp]
lib.nb_workspace_bytes.argtypes = [_i64, _i64]
lib.nb_workspace_bytes.restype = ctypes.c_size_t
lib.nb_set_workspace.argtypes = [_vp, _vp, ctypes.c_size_t]
for _f in (lib.nb_set_j, lib.nb_set_j_host):
    _f.argtypes = [_vp, _i64, _i64] + [_vp] * 14
lib.nb_update_j.argtypes = [_vp, _vp, _i64] + [_vp] * 14
lib.nb_update_j_host.argtypes = [_vp, _vp, _i64] + [_vp] * 14
lib.nb_clear.argtypes = [_vp]
lib.nb_count.argtypes = [_vp]
lib.nb_count.restype = _i64
lib.nb_set_flags.argtypes = [_vp, _vp, _vp, _i64]
lib.nb_predict.argtypes = [_vp, _dbl]
lib.nb_get_predicted.argtypes = [_vp, _i64, _i64, _vp]
for _f in (lib.nb_force, lib.nb_force_host):
    _f.argtypes = [_vp, _vp, _i64, _dbl, _vp, _vp, _vp]
lib.nb_set_tuning.argtypes = [_vp, _i32, _i32]
lib.nb_set_precision.argtypes = [_vp, _i32]
lib.nb_set_order.argtypes = [_vp, _i32]
lib.nb_force6.argtypes = [_vp, _vp, _i64, _dbl, _vp, _vp, _vp, _vp]
lib.nb_last_launch.argtypes = [_vp, ctypes.POINTER(_i64)]
lib.nb_launch_count.argtypes = [_vp]
lib.nb_launch_count.restype = _i64
lib.nb_set_profiling.argtypes = [_vp, _i32]
lib.nb_kernel_times.argtypes = [_vp, ctypes.POINTER(_dbl)]
lib.nb_sync.argtypes = [_vp]
lib.nb_strerror.argtypes = [_i32]
lib.nb_strerror.restype = ctypes.c_char_p
lib.nb_force_fused.argtypes = [_vp, _dbl, _vp, _i64, _dbl, _vp, _vp, _vp]
lib.nb_set_fused.argtypes = [_vp, _i32]
lib.nb_force_ext.argtypes = [_vp, _i64, _vp, _vp, _dbl, _vp, _vp, _vp]
lib.nb_force_ext_ids.argtypes = [_vp, _i64, _vp, _vp, _vp, _vp, _dbl, _vp, _vp, _vp]
lib.nb_set_dt.argtypes = [_vp, _i64, _i64, _vp]
lib.nb_get_state.argtypes = [_vp, _i64, _i64, _vp]
lib.nb_init_steps.argtypes = [_vp, _vp, _i64, _vp, _vp, _dbl, _dbl, _dbl]
lib.nb_next_block.argtypes = [_vp, ctypes.POINTER(_dbl), ctypes.POINTER(_i64), ctypes.POINTER(_vp)]
lib.nb_correct.argtypes = [_vp, _vp, _i64, _dbl, _vp, _vp, _dbl, _dbl, _dbl]
lib.nb_step.argtypes = [_vp, _dbl, _dbl, _dbl, _dbl, ctypes.POINTER(_dbl), ctypes.POINTER(_i64)]
lib.nb_steps.argtypes = [_vp, _i64, _dbl, _dbl, _dbl, _dbl, _dbl, _vp, _vp, _vp, ctypes.POINTER(_i64)]
lib.nb_set_steps_bound.argtypes = [_vp, _i64]
lib.nb_set_steps_queue.argtypes = [_vp, _i32]
lib.nb_block_forces.argtypes = [_vp, ctypes.POINTER(_vp), ctypes.POINTER(_vp), ctypes.POINTER(_vp)]
lib.nb_version.restype = ctypes.c_char_p
lib.nb_xchg_create.argtypes = [_vp, _i32, _i32, _i64]
lib.nb_xchg_export.argtypes = [_vp, _vp, ctypes.POINTER(_vp)]
lib.nb_xchg_attach.argtypes = [_vp, _i32, _vp, _vp]
lib.nb_xchg_destroy.argtypes = [_vp]
lib.nb_xchg_set_timeout.argtypes = [_vp, _dbl]
lib.nb_xforce.argtypes = [_vp, _i32, _i64, _vp, _vp, _vp, _vp, _dbl, _vp, _vp, _vp]
lib.nb_force_static.argtypes = [_vp, _i64, _vp, _vp, _vp, _i64, _vp, _vp, _vp, _dbl, _vp, _vp, _vp]


class NBError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        super().__init__("%s: %s (%d)" % (where, lib.nb_strerror(status).decode(), status))


def _check(status, where):
    if status != NB_OK:
        raise NBError(status, where)


def _ptr(a):
    """Address of a torch tensor / numpy array / None / int."""
    if a is None:
        return None
    if isinstance(a, int):
        return a
    if hasattr(a, "data_ptr"):
        return a.data_ptr()
    return a.ctypes.data


def nb_version():
    return lib.nb_version().decode()


def nb_strerror(status):
    return lib.nb_strerror(status).decode()


def nb_workspace_bytes(n_max, ni_max):
    return int(lib.nb_workspace_bytes(n_max, ni_max))


def nb_create(n_max, ni_max, device=0, stream=None):
    h = _vp()
    _check(lib.nb_create(ctypes.byref(h), n_max, ni_max, device, stream), "nb_create")
    return h


def nb_destroy(c):
    _check(lib.nb_destroy(c), "nb_destroy")


def nb_set_stream(c, stream):
    _check(lib.nb_set_stream(c, stream), "nb_set_stream")


def nb_set_workspace(c, dev_ptr, nbytes):
    _check(lib.nb_set_workspace(c, _ptr(dev_ptr), nbytes), "nb_set_workspace")


def _fields(m, x, v, a, j, t):
    """14 pointers from m (N,), x, v, a, j (3, N) row-contiguous (or None), t (N,) (or None)."""
    def rows(q):
        if q is None:
            return [None] * 3
        assert q.shape[0] == 3 and _contig(q)
        esz = q.element_size() if hasattr(q, "element_size") else q.itemsize
        return [_ptr(q) + r * q.shape[1] * esz for r in range(3)]
    return [_ptr(m)] + rows(x) + rows(v) + rows(a) + rows(j) + [_ptr(t)]


def _contig(q):
    return q.is_contiguous() if hasattr(q, "is_contiguous") else q.flags["C_CONTIGUOUS"]


def nb_set_j(c, first, count, m, x, v, a=None, j=None, t=None):
    """DEVICE tensors: m (count,), x, v, a, j (3, count) fp64 contiguous, t (count,)."""
    _check(lib.nb_set_j(c, first, count, *_fields(m, x, v, a, j, t)), "nb_set_j")


def nb_set_j_host(c, first, count, m, x, v, a=None, j=None, t=None):
    """HOST arrays (numpy or CPU torch tensors, ideally pinned), same shapes as nb_set_j."""
    _check(lib.nb_set_j_host(c, first, count, *_fields(m, x, v, a, j, t)), "nb_set_j_host")


def nb_update_j(c, idx, count, m, x, v, a=None, j=None, t=None):
    _check(lib.nb_update_j(c, _ptr(idx), count, *_fields(m, x, v, a, j, t)), "nb_update_j")


def nb_update_j_host(c, idx, count, m, x, v, a=None, j=None, t=None):
    """HOST idx (int32) and arrays; count <= ni_max."""
    _check(lib.nb_update_j_host(c, _ptr(idx), count, *_fields(m, x, v, a, j, t)), "nb_update_j_host")


def nb_clear(c):
    _check(lib.nb_clear(c), "nb_clear")


def nb_count(c):
    return int(lib.nb_count(c))


def nb_set_flags(c, idx, flags):
    """idx: host int32 array, flags: host uint8 array (numpy)."""
    import numpy as np
    idx = np.ascontiguousarray(idx, np.int32)
    flags = np.ascontiguousarray(flags, np.uint8)
    assert idx.shape == flags.shape
    _check(lib.nb_set_flags(c, idx.ctypes.data, flags.ctypes.data, idx.shape[0]), "nb_set_flags")


def nb_predict(c, t):
    _check(lib.nb_predict(c, float(t)), "nb_predict")


def nb_get_predicted(c, first, count, out):
    _check(lib.nb_get_predicted(c, first, count, _ptr(out)), "nb_get_predicted")


def nb_force(c, i_list, ni, eps2, acc, jrk, pot):
    """DEVICE: i_list int32 (ni,), acc, jrk fp64 (3, ni), pot fp64 (ni,) -- outputs."""
    _check(lib.nb_force(c, _ptr(i_list), ni, float(eps2), _ptr(acc), _ptr(jrk), _ptr(pot)), "nb_force")


def nb_force_host(c, i_list, ni, eps2, acc, jrk, pot):
    _check(lib.nb_force_host(c, _ptr(i_list), ni, float(eps2), _ptr(acc), _ptr(jrk), _ptr(pot)),
           "nb_force_host")


def nb_set_tuning(c, j_splits=0, reduce_mode=0):
    _check(lib.nb_set_tuning(c, j_splits, reduce_mode), "nb_set_tuning")


def nb_last_launch(c):
    out = (_i64 * 4)()
    _check(lib.nb_last_launch(c, out), "nb_last_launch")
    return {"j_splits": out[0], "ctas": out[1], "kernels": out[2], "variant": out[3]}


def nb_launch_count(c):
    return int(lib.nb_launch_count(c))


def nb_set_profiling(c, on=True):
    _check(lib.nb_set_profiling(c, 1 if on else 0), "nb_set_profiling")


NB_FUSED_MAX = 8


def nb_force_fused(c, t, i_list, ni, eps2, acc, jrk, pot):
    _check(lib.nb_force_fused(c, float(t), _ptr(i_list), ni, float(eps2), _ptr(acc), _ptr(jrk), _ptr(pot)),
           "nb_force_fused")


def nb_set_fused(c, on):
    _check(lib.nb_set_fused(c, int(bool(on))), "nb_set_fused")


def nb_force_ext(c, ni, x, v, eps2, acc, jrk, pot):
    """DEVICE x, v (3, ni) fp64 (v and jrk both None: acc + pot only)."""
    _check(lib.nb_force_ext(c, ni, _ptr(x), _ptr(v), eps2, _ptr(acc), _ptr(jrk), _ptr(pot)), "nb_force_ext")


def nb_force_ext_ids(c, ni, x, v, self_idx, iflags, eps2, acc, jrk, pot):
    """DEVICE x, v (3, ni) fp64, self_idx int32 (ni,), iflags uint8 (ni,) or None."""
    _check(lib.nb_force_ext_ids(c, ni, _ptr(x), _ptr(v), _ptr(self_idx), _ptr(iflags), eps2, _ptr(acc), _ptr(jrk),
                                _ptr(pot)), "nb_force_ext_ids")


def nb_force_static(stream, n, m, x, v, ni, xi, vi, self_idx, eps2, acc, jrk, pot):
    """No context, no allocation (nb.h): DEVICE m (n,), x, v (3, n), xi, vi (3, ni) fp64, self_idx int32
    (ni,) or None; outputs acc, jrk (3, ni) (jrk may be None), pot (ni,).  On the CURRENT device."""
    _check(lib.nb_force_static(stream, n, _ptr(m), _ptr(x), _ptr(v), ni, _ptr(xi), _ptr(vi), _ptr(self_idx), eps2,
                               _ptr(acc), _ptr(jrk), _ptr(pot)), "nb_force_static")


def nb_xchg_create(c, rank, world, ni_cap):
    _check(lib.nb_xchg_create(c, int(rank), int(world), int(ni_cap)), "nb_xchg_create")


def nb_xchg_export(c):
    """-> (handle: NB_XCHG_HANDLE_BYTES bytes for another process, dev_ptr: int for this process)."""
    buf = ctypes.create_string_buffer(NB_XCHG_HANDLE_BYTES)
    ptr = ctypes.c_void_p()
    _check(lib.nb_xchg_export(c, ctypes.cast(buf, ctypes.c_void_p), ctypes.byref(ptr)), "nb_xchg_export")
    return bytes(buf.raw), int(ptr.value)


def nb_xchg_attach(c, peer, handle=None, same_process_ptr=None):
    """handle: bytes from the peer's nb_xchg_export (another process); same_process_ptr: int."""
    buf = ctypes.create_string_buffer(bytes(handle), NB_XCHG_HANDLE_BYTES) if handle is not None else None
    _check(lib.nb_xchg_attach(c, int(peer), ctypes.cast(buf, ctypes.c_void_p) if buf is not None else None,
                              ctypes.c_void_p(same_process_ptr) if same_process_ptr is not None else None),
           "nb_xchg_attach")


def nb_xchg_set_timeout(c, seconds):
    _check(lib.nb_xchg_set_timeout(c, float(seconds)), "nb_xchg_set_timeout")


def nb_xchg_destroy(c):
    _check(lib.nb_xchg_destroy(c), "nb_xchg_destroy")


def nb_xforce(c, phase, ni, x, v, self_idx, iflags, eps2, acc, jrk, pot):
    """As nb_force_ext_ids (DEVICE pointers) plus the exchange over peer memory; phase 0, 1 or 2."""
    _check(lib.nb_xforce(c, int(phase), ni, _ptr(x), _ptr(v), _ptr(self_idx), _ptr(iflags), eps2, _ptr(acc), _ptr(jrk),
                         _ptr(pot)), "nb_xforce")


def nb_set_order(c, order):
    _check(lib.nb_set_order(c, int(order)), "nb_set_order")


def nb_force6(c, i_list, ni, eps2, acc, jrk, snp, pot):
    """DEVICE: i_list int32 (ni,); outputs acc, jrk, snp fp64 (3, ni), pot fp64 (ni,)."""
    _check(lib.nb_force6(c, _ptr(i_list), ni, float(eps2), _ptr(acc), _ptr(jrk), _ptr(snp), _ptr(pot)), "nb_force6")


def nb_set_precision(c, mode):
    _check(lib.nb_set_precision(c, int(mode)), "nb_set_precision")


def nb_set_dt(c, first, count, dt):
    _check(lib.nb_set_dt(c, first, count, _ptr(dt)), "nb_set_dt")


def nb_get_state(c, first, count, out):
    """out: DEVICE fp64 (15, count)."""
    _check(lib.nb_get_state(c, first, count, _ptr(out)), "nb_get_state")


def nb_init_steps(c, i_list, ni, acc, jrk, eta_s, dt_min, dt_max):
    _check(lib.nb_init_steps(c, _ptr(i_list), ni, _ptr(acc), _ptr(jrk), eta_s, dt_min, dt_max),
           "nb_init_steps")


def nb_next_block(c):
    """Returns (t_next, ni, device address of the context-owned int32 list)."""
    t, ni, lst = _dbl(0.0), _i64(0), _vp()
    _check(lib.nb_next_block(c, ctypes.byref(t), ctypes.byref(ni), ctypes.byref(lst)), "nb_next_block")
    return t.value, ni.value, lst.value


def nb_correct(c, i_list, ni, t1, acc, jrk, eta, dt_min, dt_max):
    _check(lib.nb_correct(c, _ptr(i_list), ni, t1, _ptr(acc), _ptr(jrk), eta, dt_min, dt_max), "nb_correct")


def nb_step(c, eps2, eta, dt_min, dt_max):
    """One block step on the device; returns (t, ni)."""
    t, ni = _dbl(0.0), _i64(0)
    _check(lib.nb_step(c, eps2, eta, dt_min, dt_max, ctypes.byref(t), ctypes.byref(ni)), "nb_step")
    return t.value, ni.value


def nb_steps(c, k, eps2, eta, dt_min, dt_max, t_end=float("inf"), log=True, times=False):
    """Up to k block steps on the device; returns (done, t_log, ni_log) -- numpy arrays of length
    done (None, None with log=False) -- and with times=True also the device time of every step in
    microseconds."""
    import numpy as np
    done = _i64(0)
    t_log = np.empty(max(k, 1), np.float64) if log else None
    ni_log = np.empty(max(k, 1), np.int64) if log else None
    us_log = np.empty(max(k, 1), np.float64) if times else None
    _check(lib.nb_steps(c, k, eps2, eta, dt_min, dt_max, t_end, _ptr(t_log), _ptr(ni_log), _ptr(us_log),
                        ctypes.byref(done)), "nb_steps")
    d = done.value
    out = (d, t_log[:d] if log else None, ni_log[:d] if log else None)
    return out + (us_log[:d],) if times else out


def nb_set_steps_bound(c, max_pairs):
    _check(lib.nb_set_steps_bound(c, int(max_pairs)), "nb_set_steps_bound")


def nb_set_steps_queue(c, on):
    _check(lib.nb_set_steps_queue(c, int(on)), "nb_set_steps_queue")


def nb_block_forces(c):
    """Device addresses (acc, jrk, pot) of the last nb_step's forces."""
    a, j, p = _vp(), _vp(), _vp()
    _check(lib.nb_block_forces(c, ctypes.byref(a), ctypes.byref(j), ctypes.byref(p)), "nb_block_forces")
    return a.value, j.value, p.value


def nb_kernel_times(c):
    """Totals since profiling was switched on (after a stream sync): summed ms and launch counts
    of the predictor / pair / reduction kernels."""
    out = (_dbl * 6)()
    _check(lib.nb_kernel_times(c, out), "nb_kernel_times")
    return {"predict_ms": out[0], "pair_ms": out[1], "reduce_ms": out[2],
            "n_predict": int(out[3]), "n_pair": int(out[4]), "n_reduce": int(out[5])}


def nb_sync(c):
    _check(lib.nb_sync(c), "nb_sync")
