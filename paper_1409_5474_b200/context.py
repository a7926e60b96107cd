"""Convenience wrapper: one nb context + torch-allocated outputs.  Marshalling only."""
import torch

from . import binding as nb


class _DeviceView:
    """A context-owned device array seen through __cuda_array_interface__ (no copy)."""

    def __init__(self, ptr, n, typestr):
        self.__cuda_array_interface__ = {"shape": (int(n),), "typestr": typestr,
                                         "data": (int(ptr), False), "version": 2}


class Context:
    def __init__(self, n_max, ni_max=None, device=0, stream=None):
        self.device = torch.device("cuda", device)
        self.n_max = int(n_max)
        self.ni_max = int(ni_max if ni_max is not None else n_max)
        if stream is None:
            stream = torch.cuda.current_stream(self.device).cuda_stream
        self.h = nb.nb_create(self.n_max, self.ni_max, device, stream)

    def close(self):
        if self.h is not None:
            nb.nb_destroy(self.h)
            self.h = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- j-set ------------------------------------------------------------------------------
    def _dev(self, q, dtype=torch.float64):
        if q is None:
            return None
        return torch.as_tensor(q, dtype=dtype).to(self.device).contiguous()

    def set_j(self, m, x, v, a=None, j=None, t=None, first=0):
        """Arrays of any kind (numpy / torch, host or device); copied to the device by torch,
        then handed to nb_set_j as device pointers."""
        d = [self._dev(q) for q in (m, x, v, a, j, t)]
        nb.nb_set_j(self.h, first, d[0].shape[0], *d)
        self._keep = d   # alive until the stream has consumed them

    def update_j(self, idx, m, x, v, a=None, j=None, t=None):
        i = self._dev(idx, torch.int32)
        d = [self._dev(q) for q in (m, x, v, a, j, t)]
        nb.nb_update_j(self.h, i, i.shape[0], *d)
        self._keep = [i] + d

    def load_case(self, case):
        self.set_j(case.m, case.x, case.v, case.a, case.j, case.t)
        fl = case.flags.nonzero()[0]
        if fl.size:
            nb.nb_set_flags(self.h, fl, case.flags[fl])

    def set_flags(self, idx, flags):
        nb.nb_set_flags(self.h, idx, flags)

    # -- predictor / force --------------------------------------------------------------------
    def predict(self, t):
        nb.nb_predict(self.h, t)

    def predicted(self, first=0, count=None):
        count = nb.nb_count(self.h) - first if count is None else count
        out = torch.empty((6, count), dtype=torch.float64, device=self.device)
        nb.nb_get_predicted(self.h, first, count, out)
        return out[:3], out[3:]

    def force(self, i_list, eps2):
        il = self._dev(i_list, torch.int32)
        ni = il.shape[0]
        acc = torch.empty((3, ni), dtype=torch.float64, device=self.device)
        jrk = torch.empty((3, ni), dtype=torch.float64, device=self.device)
        pot = torch.empty((ni,), dtype=torch.float64, device=self.device)
        nb.nb_force(self.h, il, ni, eps2, acc, jrk, pot)
        self._keep_i = il
        return acc, jrk, pot

    def order(self, order):
        """4 (default) or 6: the predictor then also writes the records nb_force6 streams."""
        nb.nb_set_order(self.h, order)

    def force6(self, i_list, eps2):
        il = self._dev(i_list, torch.int32)
        ni = il.shape[0]
        out = [torch.empty((3, ni), dtype=torch.float64, device=self.device) for _ in range(3)]
        pot = torch.empty((ni,), dtype=torch.float64, device=self.device)
        nb.nb_force6(self.h, il, ni, eps2, out[0], out[1], out[2], pot)
        self._keep_i = il
        return out[0], out[1], out[2], pot

    def precision(self, mode):
        """0 = mixed (48-bit differences, fp32 pair terms), 1 = IEEE double throughout."""
        nb.nb_set_precision(self.h, mode)

    def tuning(self, j_splits=0, reduce_mode=0):
        nb.nb_set_tuning(self.h, j_splits, reduce_mode)

    def last_launch(self):
        return nb.nb_last_launch(self.h)

    def sync(self):
        nb.nb_sync(self.h)

    # -- host-buffer entry points (the end-to-end path: copies are part of the call) ----------
    def set_j_host(self, m, x, v, a=None, j=None, t=None, first=0):
        """HOST arrays (numpy or pinned CPU tensors), fp64 contiguous; staged by the library."""
        nb.nb_set_j_host(self.h, first, m.shape[0], m, x, v, a, j, t)
        self._keep_host = [m, x, v, a, j, t]     # pinned sources are read later, on the stream

    def update_j_host(self, idx, m, x, v, a=None, j=None, t=None):
        """HOST int32 idx and HOST fp64 arrays of the idx.shape[0] updated particles."""
        nb.nb_update_j_host(self.h, idx, idx.shape[0], m, x, v, a, j, t)
        self._keep_host = [idx, m, x, v, a, j, t]

    def force_host(self, i_list, eps2, acc, jrk, pot):
        """HOST int32 i_list and HOST fp64 outputs acc, jrk (3, ni), pot (ni,); returns after
        the results are back on the host."""
        nb.nb_force_host(self.h, i_list, i_list.shape[0], eps2, acc, jrk, pot)

    def force_fused(self, t, i_list, eps2):
        """Forces at time t on <= NB_FUSED_MAX members of the j-set, predictor fused in (one pass)."""
        il = self._dev(i_list, torch.int32)
        ni = il.shape[0]
        acc = torch.empty((3, ni), dtype=torch.float64, device=self.device)
        jrk = torch.empty((3, ni), dtype=torch.float64, device=self.device)
        pot = torch.empty((ni,), dtype=torch.float64, device=self.device)
        nb.nb_force_fused(self.h, t, il, ni, eps2, acc, jrk, pot)
        self._keep = [il]
        return acc, jrk, pot

    def fused(self, on=True):
        nb.nb_set_fused(self.h, on)

    def force_ext(self, x, v, eps2):
        """Forces on particles given by value: x, v (3, ni) of any kind; v None -> (acc, None, pot)."""
        dx = self._dev(x)
        dv = self._dev(v)
        ni = dx.shape[1]
        acc = torch.empty((3, ni), dtype=torch.float64, device=self.device)
        jrk = torch.empty((3, ni), dtype=torch.float64, device=self.device) if dv is not None else None
        pot = torch.empty((ni,), dtype=torch.float64, device=self.device)
        nb.nb_force_ext(self.h, ni, dx, dv, eps2, acc, jrk, pot)
        self._keep = [dx, dv]
        return acc, jrk, pot

    def force_ext_ids(self, x, v, self_idx, iflags, eps2):
        """By value, with the index of the j-set member each i-particle is (or -1) and its flag."""
        dx, dv = self._dev(x), self._dev(v)
        ds = self._dev(self_idx, torch.int32)
        df = self._dev(iflags, torch.uint8) if iflags is not None else None
        ni = dx.shape[1]
        acc = torch.empty((3, ni), dtype=torch.float64, device=self.device)
        jrk = torch.empty((3, ni), dtype=torch.float64, device=self.device)
        pot = torch.empty((ni,), dtype=torch.float64, device=self.device)
        nb.nb_force_ext_ids(self.h, ni, dx, dv, ds, df, eps2, acc, jrk, pot)
        self._keep = [dx, dv, ds, df]
        return acc, jrk, pot

    # -- j-sharding with the exchange done by the kernels over peer memory (nb.h: nb_xforce) -----
    def xchg_create(self, rank, world, ni_cap):
        nb.nb_xchg_create(self.h, rank, world, ni_cap)

    def xchg_export(self):
        """(IPC handle bytes for another process, device address for another context of this one)."""
        return nb.nb_xchg_export(self.h)

    def xchg_attach(self, peer, handle=None, same_process_ptr=None):
        nb.nb_xchg_attach(self.h, peer, handle, same_process_ptr)

    def xchg_timeout(self, seconds):
        nb.nb_xchg_set_timeout(self.h, seconds)

    def xchg_destroy(self):
        nb.nb_xchg_destroy(self.h)

    def xforce(self, x, v, self_idx, iflags, eps2, phase=0, out=None):
        """force_ext_ids on this rank's j-slice + the exchange: phase 0 = complete forces; 1 = compute
        and push (returns this rank's partial forces); 2 = wait and sum into `out` (the tensors phase
        1 returned)."""
        if phase == 2:
            acc, jrk, pot = out
            nb.nb_xforce(self.h, 2, pot.shape[0], None, None, None, None, eps2, acc, jrk, pot)
            return acc, jrk, pot
        dx, dv = self._dev(x), self._dev(v)
        ds = self._dev(self_idx, torch.int32)
        df = self._dev(iflags, torch.uint8) if iflags is not None else None
        ni = dx.shape[1]
        acc = torch.empty((3, ni), dtype=torch.float64, device=self.device)
        jrk = torch.empty((3, ni), dtype=torch.float64, device=self.device)
        pot = torch.empty((ni,), dtype=torch.float64, device=self.device)
        nb.nb_xforce(self.h, phase, ni, dx, dv, ds, df, eps2, acc, jrk, pot)
        self._keep = [dx, dv, ds, df]
        return acc, jrk, pot

    # -- block-step layer (marshalling only) --------------------------------------------------
    def init_steps(self, i_list, acc, jrk, eta_s, dt_min, dt_max):
        il = self._dev(i_list, torch.int32)
        nb.nb_init_steps(self.h, il, il.shape[0], acc, jrk, eta_s, dt_min, dt_max)
        self._keep = [il, acc, jrk]

    def set_dt(self, dt, first=0):
        d = self._dev(dt)
        nb.nb_set_dt(self.h, first, d.shape[0], d)
        self._keep = [d]

    def state(self, first=0, count=None):
        """(15, count) fp64 device tensor: the 14 stored fields, then dt."""
        count = nb.lib.nb_count(self.h) - first if count is None else count
        out = torch.empty((15, count), dtype=torch.float64, device=self.device)
        nb.nb_get_state(self.h, first, count, out)
        return out

    def next_block(self):
        """(t_next, ni, int32 device tensor viewing the context-owned list of due particles)."""
        t, ni, addr = nb.nb_next_block(self.h)
        if ni == 0:
            return t, ni, torch.empty(0, dtype=torch.int32, device=self.device)
        return t, ni, torch.as_tensor(_DeviceView(addr, ni, "<i4"), device=self.device)

    def correct(self, i_list, t1, acc, jrk, eta, dt_min, dt_max):
        il = self._dev(i_list, torch.int32)
        nb.nb_correct(self.h, il, il.shape[0], t1, acc, jrk, eta, dt_min, dt_max)
        self._keep = [il, acc, jrk]

    def step(self, eps2, eta, dt_min, dt_max):
        return nb.nb_step(self.h, eps2, eta, dt_min, dt_max)

    def steps(self, k, eps2, eta, dt_min, dt_max, t_end=float("inf"), log=True, times=False):
        """Up to k block steps without a host round trip per step: (done, t_log, ni_log[, us_log])."""
        return nb.nb_steps(self.h, k, eps2, eta, dt_min, dt_max, t_end, log, times)

    def steps_bound(self, max_pairs):
        nb.nb_set_steps_bound(self.h, max_pairs)

    def steps_queue(self, on):
        nb.nb_set_steps_queue(self.h, on)

    # -- measurement --------------------------------------------------------------------------
    def profiling(self, on=True):
        nb.nb_set_profiling(self.h, on)

    def kernel_times(self):
        return nb.nb_kernel_times(self.h)

    def launch_count(self):
        return nb.nb_launch_count(self.h)
