"""Thin ctypes binding of libfh_b200.so (include/fh_b200.h): argument marshalling only.

Every step of the hot path runs inside the library's CUDA kernels; PyTorch is used here for
device memory (the HBM arena, vectors) and streams, nothing else.  There is no CPU fallback:
importing this module fails if the shared library is missing, and every call raises FhError on
a non-zero return code.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfh_b200.so")
if not os.path.exists(LIB_PATH):
    raise ImportError("libfh_b200.so is not built: run `python -m paper_2606_04771_b200.build` "
                      "(or __graft_entry__.build()); there is no CPU fallback")
lib = C.CDLL(LIB_PATH)

c_int, c_i64, c_dbl, c_void_p, c_size_t = C.c_int, C.c_int64, C.c_double, C.c_void_p, C.c_size_t
P = C.POINTER


class fh_params(C.Structure):
    _fields_ = [("krylov_dim", c_int), ("krylov_tol", c_dbl), ("chi_max_full", c_int), ("eps_trunc", c_dbl),
                ("krylov_adapt_tol", c_dbl)]


_SIGS = {
    "fh_ctx_create": (c_int, [P(c_void_p), c_void_p, c_void_p, c_size_t]),
    "fh_ctx_destroy": (None, [c_void_p]),
    "fh_last_error": (C.c_char_p, [c_void_p]),
    "fh_arena_stats": (c_int, [c_void_p, P(c_size_t), P(c_size_t)]),
    "fh_set_option": (c_int, [c_void_p, c_int, c_int]),
    "fh_canonical_weight": (c_dbl, [c_int, c_int]),
    "fh_host_set_symmetry": (c_int, [c_int]),
    "fh_mpo_build": (c_int, [c_void_p, c_int, c_dbl, c_dbl, P(c_void_p)]),
    "fh_mpo_destroy": (None, [c_void_p]),
    "fh_mpo_get_site": (c_int, [c_void_p, c_int, c_void_p, c_void_p]),
    "mps_init_neel": (c_int, [c_void_p, c_void_p, c_int, P(c_void_p)]),
    "mps_create": (c_int, [c_void_p, c_int, P(c_void_p)]),
    "mps_destroy": (None, [c_void_p, c_void_p]),
    "mps_set_bond": (c_int, [c_void_p, c_void_p, c_int, c_int, c_void_p, c_void_p, c_void_p]),
    "mps_get_bond": (c_int, [c_void_p, c_int, P(c_int), c_void_p, c_void_p, c_void_p]),
    "mps_site_layout": (c_int, [c_void_p, c_int, P(c_int), P(c_i64), c_void_p, c_void_p]),
    "mps_set_site": (c_int, [c_void_p, c_void_p, c_int, c_void_p, c_int]),
    "mps_get_site": (c_int, [c_void_p, c_void_p, c_int, c_void_p, c_i64, c_int]),
    "mps_get_svals": (c_int, [c_void_p, c_int, P(c_int), c_void_p]),
    "fh_dmma_peak_tflops": (c_int, [c_void_p, c_int, P(c_dbl)]),
    "fh_vec_kernels_gbs": (c_int, [c_void_p, c_i64, c_int, c_int, P(c_dbl)]),
    "fh_vec_wdot": (c_int, [c_void_p, c_i64, c_int, c_void_p, c_void_p, c_void_p, c_void_p, P(c_dbl)]),
    "fh_static_setup": (c_int, []),
    "fh_vec_wdot_static": (c_int, [c_i64, c_int, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p]),
    "fh_static_last_error": (C.c_char_p, []),
    "fh_vec_lanczos_update": (c_int, [c_void_p, c_i64, c_int, c_void_p, c_void_p, c_dbl, c_dbl, c_dbl, c_dbl, c_void_p,
                                      c_void_p, c_void_p, P(c_dbl)]),
    "fh_zgemm_split": (c_int, [c_void_p, c_int, c_int, c_int, c_void_p, c_void_p, c_int, c_void_p, c_void_p, c_void_p, c_void_p,
                               c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_int]),
    "fh_vec_lincomb": (c_int, [c_void_p, c_i64, c_int, c_void_p, c_void_p, c_i64, c_void_p]),
    "fh_copy_blocks": (c_int, [c_void_p, c_int, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p,
                               c_void_p, c_void_p]),
    "mps_drop_site": (c_int, [c_void_p, c_void_p, c_int]),
    "heff_apply_host": (c_int, [c_void_p, c_void_p, c_void_p]),
    "env_update_left": (c_int, [c_void_p, c_void_p, c_void_p, c_int]),
    "env_update_right": (c_int, [c_void_p, c_void_p, c_void_p, c_int]),
    "env_layout": (c_int, [c_void_p, c_int, c_int, P(c_int), P(c_i64), c_void_p, c_void_p]),
    "env_get": (c_int, [c_void_p, c_void_p, c_int, c_int, c_void_p, c_i64, c_int]),
    "env_set": (c_int, [c_void_p, c_void_p, c_int, c_int, c_int, c_void_p, c_void_p, c_int]),
    "heff_plan": (c_int, [c_void_p, c_void_p, c_void_p, c_int, c_int]),
    "heff_layout": (c_int, [c_void_p, P(c_int), P(c_i64), c_void_p, c_void_p]),
    "heff_get_tasks": (c_int, [c_void_p, c_int, P(c_int), P(c_int), c_void_p, c_void_p]),
    "heff_apply": (c_int, [c_void_p, c_void_p, c_void_p]),
    "heff_import": (c_int, [c_void_p, c_void_p, c_void_p]),
    "heff_export": (c_int, [c_void_p, c_void_p, c_void_p]),
    "heff_flops": (c_i64, [c_void_p]),
    "heff_inner": (c_int, [c_void_p, c_void_p, c_void_p, P(c_dbl)]),
    "heff_expm": (c_int, [c_void_p, c_void_p, c_void_p, c_dbl, c_int]),
    "heff_expm_adaptive": (c_int, [c_void_p, c_void_p, c_void_p, c_dbl, c_int, c_dbl, P(c_int)]),
    "fh_krylov_stats": (c_int, [c_void_p, P(C.c_int64), P(C.c_int64)]),
    "fh_factorization_stats": (c_int, [c_void_p, P(C.c_int64)]),
    "fh_plan_cache_stats": (c_int, [c_void_p, P(C.c_int64), P(C.c_int64), P(C.c_int64)]),
    "fh_plan_cache_limit": (c_int, [c_void_p, C.c_int64]),
    "mps_save": (c_int, [c_void_p, c_void_p, C.c_char_p]),
    "mps_load": (c_int, [c_void_p, c_void_p, C.c_char_p, P(c_void_p)]),
    "tdvp2_sweep": (c_int, [c_void_p, c_void_p, c_void_p, c_dbl, P(fh_params)]),
    "tdvp1_sweep": (c_int, [c_void_p, c_void_p, c_void_p, c_dbl, P(fh_params)]),
    "tdvp_sweep_auto": (c_int, [c_void_p, c_void_p, c_void_p, c_dbl, P(fh_params), P(c_int)]),
    "tdvp2_last_stats": (c_int, [c_void_p, P(c_dbl), P(c_int), P(c_int), P(c_int)]),
    "measure_local": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p]),
    "measure_global": (c_int, [c_void_p, c_void_p, c_void_p, P(c_dbl), P(c_dbl)]),
    "fh_get_timers": (c_int, [c_void_p, P(c_dbl), P(c_dbl), P(c_dbl), P(c_dbl), P(c_dbl)]),
    "fh_reset_timers": (c_int, [c_void_p]),
    "fh_get_traffic": (c_int, [c_void_p, P(c_i64), P(c_i64)]),
    "fh_enable_timers": (c_int, [c_void_p, c_int]),
    "fh_launch_count": (c_i64, [c_void_p]),
    "fh_cublas_gemm_seconds": (c_int, [c_void_p, c_int, c_int, c_int, P(c_dbl)]),
    "fh_coef_left": (c_dbl, [c_int] * 9),
    "fh_coef_right": (c_dbl, [c_int] * 9),
    "fh_host_plan": (c_int, [c_int, c_int, c_dbl, c_dbl, c_int, c_void_p, c_int, c_void_p, c_int, c_void_p,
                             c_int, c_void_p]),
    "fh_host_get_tasks": (c_int, [c_int, P(c_int), P(c_int), c_void_p, c_void_p, P(c_i64)]),
    "fh_host_get_units": (c_int, [c_int, P(c_int), c_void_p, P(c_int), c_void_p, P(c_i64)]),
    "fh_host_get_tc_tiles": (c_int, [c_int, c_int, c_int, P(c_int), c_void_p, c_void_p, P(c_int), P(c_int), c_void_p, c_void_p,
                                     P(c_i64)]),
}
EXPORTS = sorted(_SIGS)
for _name, (_res, _args) in _SIGS.items():
    _f = getattr(lib, _name)
    _f.restype = _res
    _f.argtypes = _args


class FhError(RuntimeError):
    pass


def _np_ptr(a):
    return a.ctypes.data_as(c_void_p)


def _i32(x):
    return np.ascontiguousarray(np.asarray(x, dtype=np.int32))


# ------------------------------------------------------------------ host-only entry points
def fh_canonical_weight(c, b):
    """Metric of a right-canonical site tensor as the LIBRARY defines it (labels (q, tj))."""
    return lib.fh_canonical_weight(int(c[1]), int(b[1]))


# ------------------------------------------------------------------ allocation-free entry point (no context)
STATIC_MAX_BLOCKS, STATIC_MAX_ELEMS, STATIC_SCRATCH_BYTES = 16384, 1 << 32, 196872


def fh_static_setup():
    rc = lib.fh_static_setup()
    if rc != 0:
        raise FhError("fh_static_setup: rc=%d: %s" % (rc, lib.fh_static_last_error().decode()))


def fh_vec_wdot_static(n, nblk, blk_len_dev, blk_weight_dev, x, y, result, stream=None):
    """blk_len_dev (int64), blk_weight_dev (int32), x, y (complex128), result (2 float64): CUDA tensors; the call
    only launches (no synchronisation): read `result` after synchronising the stream."""
    rc = lib.fh_vec_wdot_static(int(n), int(nblk), c_void_p(blk_len_dev.data_ptr()), c_void_p(blk_weight_dev.data_ptr()),
                                c_void_p(x.data_ptr()), c_void_p(y.data_ptr()), c_void_p(result.data_ptr()),
                                c_void_p(stream if stream else 0))
    if rc != 0:
        raise FhError("fh_vec_wdot_static: rc=%d: %s" % (rc, lib.fh_static_last_error().decode()))


def fh_coef_left(*t):
    return lib.fh_coef_left(*[int(x) for x in t])


def fh_coef_right(*t):
    return lib.fh_coef_right(*[int(x) for x in t])


def fh_host_plan(site, nsite, t_h, U, dims_l, dims_r, L_keys, R_keys):
    """dims_*: {(q,tj): d}; *_keys: canonical-order env keys ((q',tj'), w, (q,tj)).  Returns
    [(tuples int32[n,3], alpha f64[n], nout, flops)] for stage 1 and 2."""
    bl = _i32([[q, tj, d] for (q, tj), d in sorted(dims_l.items())])
    br = _i32([[q, tj, d] for (q, tj), d in sorted(dims_r.items())])
    Ll = _i32([[xp[0], xp[1], w, x[0], x[1]] for xp, w, x in L_keys])
    Rl = _i32([[xp[0], xp[1], w, x[0], x[1]] for xp, w, x in R_keys])
    rc = lib.fh_host_plan(site, nsite, t_h, U, len(bl), _np_ptr(bl), len(br), _np_ptr(br),
                          len(Ll), _np_ptr(Ll), len(Rl), _np_ptr(Rl))
    if rc != 0:
        raise FhError("fh_host_plan failed: %d" % rc)
    out = []
    for stage in (1, 2):
        nt, no, fl = c_int(), c_int(), c_i64()
        lib.fh_host_get_tasks(stage, C.byref(nt), C.byref(no), None, None, C.byref(fl))
        tup = np.zeros((nt.value, 3), dtype=np.int32)
        al = np.zeros(nt.value, dtype=np.float64)
        lib.fh_host_get_tasks(stage, C.byref(nt), C.byref(no), _np_ptr(tup), _np_ptr(al), C.byref(fl))
        out.append((tup, al, no.value, fl.value))
    return out


def fh_host_get_tc_tiles(stage, grid, static_side):
    """(tiles int32[n,6], cta_begin int32[grid+1], seg_img int64[nseg], seg_operand int64[nseg], image chunks, image bytes)."""
    nt, ns, nc, nb = c_int(), c_int(), c_int(), c_i64()
    rc = lib.fh_host_get_tc_tiles(stage, grid, 0, C.byref(nt), None, None, C.byref(ns), None, None, None, None)
    if rc != 0:
        raise FhError("fh_host_get_tc_tiles failed: %d" % rc)
    tiles = np.zeros((nt.value, 6), dtype=np.int32)
    cb = np.zeros(grid + 1, dtype=np.int32)
    img, opd = np.zeros(ns.value, dtype=np.int64), np.zeros(ns.value, dtype=np.int64)
    rc = lib.fh_host_get_tc_tiles(stage, grid, static_side, C.byref(nt), _np_ptr(tiles), _np_ptr(cb), C.byref(ns), C.byref(nc),
                                  _np_ptr(img), _np_ptr(opd), C.byref(nb))
    if rc != 0:
        raise FhError("fh_host_get_tc_tiles failed: %d" % rc)
    return tiles, cb, img, opd, nc.value, nb.value


def fh_host_get_units(stage):
    """Warp-unit list of the last fh_host_plan: (units int32[n,6] = out, m0, n0, mt, nt, steps;
    outs int32[nout,3] = M, N, steps; dmma_padded)."""
    nu, no, dp = c_int(), c_int(), c_i64()
    lib.fh_host_get_units(stage, C.byref(nu), None, C.byref(no), None, C.byref(dp))
    units = np.zeros((nu.value, 6), dtype=np.int32)
    outs = np.zeros((no.value, 3), dtype=np.int32)
    rc = lib.fh_host_get_units(stage, C.byref(nu), _np_ptr(units), C.byref(no), _np_ptr(outs), C.byref(dp))
    if rc != 0:
        raise FhError("fh_host_get_units failed: %d" % rc)
    return units, outs, dp.value


# ------------------------------------------------------------------ device objects
class Context:
    """fh_ctx: owns the HBM arena (a torch uint8 tensor) and the stream."""

    def __init__(self, arena_bytes, stream=None, device="cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise FhError("no CUDA device: the library has no CPU path")
        self.torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.arena = torch.empty(int(arena_bytes), dtype=torch.uint8, device=self.device)
        h = c_void_p()
        rc = lib.fh_ctx_create(C.byref(h), c_void_p(self.stream.cuda_stream), c_void_p(self.arena.data_ptr()),
                               c_size_t(int(arena_bytes)))
        if rc != 0:
            raise FhError("fh_ctx_create failed: %d" % rc)
        self.h = h

    def check(self, rc, what=""):
        if rc != 0:
            msg = lib.fh_last_error(self.h)
            raise FhError("%s failed (%d): %s" % (what, rc, msg.decode() if msg else ""))

    def close(self):
        if self.h:
            lib.fh_ctx_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # --- model / state
    def fh_mpo_build(self, L, t_h, U):
        h = c_void_p()
        self.check(lib.fh_mpo_build(self.h, L, t_h, U, C.byref(h)), "fh_mpo_build")
        return h

    def fh_mpo_get_site(self, mpo, site):
        val = np.zeros((6, 6, 4, 4))
        rank2 = np.zeros((6, 6), dtype=np.int32)
        self.check(lib.fh_mpo_get_site(mpo, site, _np_ptr(val), _np_ptr(rank2)), "fh_mpo_get_site")
        return val, rank2

    def mps_init_neel(self, mpo, L):
        h = c_void_p()
        self.check(lib.mps_init_neel(self.h, mpo, L, C.byref(h)), "mps_init_neel")
        return h

    def mps_create(self, L):
        h = c_void_p()
        self.check(lib.mps_create(self.h, L, C.byref(h)), "mps_create")
        return h

    def mps_destroy(self, mps):
        lib.mps_destroy(self.h, mps)

    def mps_set_bond(self, mps, bond, dims):
        items = sorted(dims.items())
        q, tj, d = _i32([k[0] for k, _ in items]), _i32([k[1] for k, _ in items]), _i32([v for _, v in items])
        self.check(lib.mps_set_bond(self.h, mps, bond, len(items), _np_ptr(q), _np_ptr(tj), _np_ptr(d)), "mps_set_bond")

    def mps_get_bond(self, mps, bond):
        n = c_int()
        self.check(lib.mps_get_bond(mps, bond, C.byref(n), None, None, None), "mps_get_bond")
        q, tj, d = (np.zeros(n.value, dtype=np.int32) for _ in range(3))
        self.check(lib.mps_get_bond(mps, bond, C.byref(n), _np_ptr(q), _np_ptr(tj), _np_ptr(d)), "mps_get_bond")
        return {(int(a), int(b)): int(c) for a, b, c in zip(q, tj, d)}

    def _layout(self, fn, nlab, *args):
        nb, ne = c_int(), c_i64()
        rc = fn(*args, C.byref(nb), C.byref(ne), None, None)
        self.check(rc, fn.__name__)
        lab = np.zeros((nb.value, nlab), dtype=np.int32)
        dims = np.zeros((nb.value, 2), dtype=np.int32)
        self.check(fn(*args, C.byref(nb), C.byref(ne), _np_ptr(lab), _np_ptr(dims)), fn.__name__)
        return lab, dims, ne.value

    def mps_site_layout(self, mps, site):
        return self._layout(lib.mps_site_layout, 5, mps, site)

    def env_layout(self, mps, which, bond):
        return self._layout(lib.env_layout, 5, mps, which, bond)

    def heff_layout(self, nsite):
        return self._layout(lib.heff_layout, 8 if nsite == 2 else 5, self.h)

    def mps_set_site(self, mps, site, data):
        """data: numpy complex128 1-D (host) or torch complex128 CUDA tensor, blocks back to back."""
        if isinstance(data, np.ndarray):
            data = np.ascontiguousarray(data, dtype=np.complex128)
            self.check(lib.mps_set_site(self.h, mps, site, _np_ptr(data), 0), "mps_set_site")
        else:
            self.check(lib.mps_set_site(self.h, mps, site, c_void_p(data.data_ptr()), 1), "mps_set_site")

    def mps_get_site(self, mps, site):
        _, _, ne = self.mps_site_layout(mps, site)
        out = np.zeros(ne, dtype=np.complex128)
        self.check(lib.mps_get_site(self.h, mps, site, _np_ptr(out), out.size, 0), "mps_get_site")
        return out

    def mps_get_svals(self, mps, bond):
        """{(q,tj): kept singular values (descending)} of the last SVD split on `bond`."""
        n = c_int()
        self.check(lib.mps_get_svals(mps, bond, C.byref(n), None), "mps_get_svals")
        s = np.zeros(n.value)
        self.check(lib.mps_get_svals(mps, bond, C.byref(n), _np_ptr(s)), "mps_get_svals")
        out, o = {}, 0
        for sec, d in self.mps_get_bond(mps, bond).items():
            out[sec] = s[o:o + d]
            o += d
        return out if n.value else {}

    def fh_dmma_peak_tflops(self, reps=5):
        t = c_dbl()
        self.check(lib.fh_dmma_peak_tflops(self.h, reps, C.byref(t)), "fh_dmma_peak_tflops")
        return t.value

    def fh_vec_kernels_gbs(self, n_elems, m=10, reps=10):
        g = (c_dbl * 7)()
        self.check(lib.fh_vec_kernels_gbs(self.h, int(n_elems), int(m), int(reps), g), "fh_vec_kernels_gbs")
        return dict(zip(("wdot", "axpy", "scale", "lincomb", "pack", "pack_transposed", "lanczos_update"),
                        [float(v) for v in g]))

    def mps_save(self, mps, path):
        self.check(lib.mps_save(self.h, mps, os.fsencode(path)), "mps_save")

    def mps_load(self, mpo, path):
        h = c_void_p()
        self.check(lib.mps_load(self.h, mpo, os.fsencode(path), C.byref(h)), "mps_load")
        return h

    def mps_drop_site(self, mps, site):
        self.check(lib.mps_drop_site(self.h, mps, site), "mps_drop_site")

    def heff_apply_host(self, theta, out):
        """theta, out: host buffers (numpy complex128 or pinned torch CPU tensors)."""
        pi = theta.ctypes.data if isinstance(theta, np.ndarray) else theta.data_ptr()
        po = out.ctypes.data if isinstance(out, np.ndarray) else out.data_ptr()
        self.check(lib.heff_apply_host(self.h, c_void_p(pi), c_void_p(po)), "heff_apply_host")

    def env_update_left(self, mpo, mps, site):
        self.check(lib.env_update_left(self.h, mpo, mps, site), "env_update_left")

    def env_update_right(self, mpo, mps, site):
        self.check(lib.env_update_right(self.h, mpo, mps, site), "env_update_right")

    def env_get(self, mps, which, bond):
        lab, dims, ne = self.env_layout(mps, which, bond)
        out = np.zeros(ne, dtype=np.complex128)
        self.check(lib.env_get(self.h, mps, which, bond, _np_ptr(out), out.size, 0), "env_get")
        return lab, dims, out

    def env_set(self, mps, which, bond, labels, data):
        labels = _i32(labels)
        if isinstance(data, np.ndarray):
            data = np.ascontiguousarray(data, dtype=np.complex128)
            self.check(lib.env_set(self.h, mps, which, bond, len(labels), _np_ptr(labels), _np_ptr(data), 0), "env_set")
        else:
            self.check(lib.env_set(self.h, mps, which, bond, len(labels), _np_ptr(labels),
                                   c_void_p(data.data_ptr()), 1), "env_set")

    # --- hot path
    def heff_plan(self, mpo, mps, site, nsite):
        self.check(lib.heff_plan(self.h, mpo, mps, site, nsite), "heff_plan")

    def heff_get_tasks(self, stage):
        nt, no = c_int(), c_int()
        self.check(lib.heff_get_tasks(self.h, stage, C.byref(nt), C.byref(no), None, None), "heff_get_tasks")
        tup = np.zeros((nt.value, 3), dtype=np.int32)
        al = np.zeros(nt.value, dtype=np.float64)
        self.check(lib.heff_get_tasks(self.h, stage, C.byref(nt), C.byref(no), _np_ptr(tup), _np_ptr(al)), "heff_get_tasks")
        return tup, al, no.value

    def heff_apply(self, theta, out):
        """theta, out: torch complex128 CUDA tensors (device pointers are passed through)."""
        self.check(lib.heff_apply(self.h, c_void_p(theta.data_ptr()), c_void_p(out.data_ptr())), "heff_apply")

    def heff_import(self, blocks, vec):
        """interchange format (blocks back to back, heff_layout order) -> planned layout; CUDA tensors."""
        self.check(lib.heff_import(self.h, c_void_p(blocks.data_ptr()), c_void_p(vec.data_ptr())), "heff_import")

    def heff_export(self, vec, blocks):
        """planned layout -> interchange format; CUDA tensors."""
        self.check(lib.heff_export(self.h, c_void_p(vec.data_ptr()), c_void_p(blocks.data_ptr())), "heff_export")

    def fh_vec_wdot(self, blk_len, blk_weight, x, y):
        bl, bw = np.ascontiguousarray(blk_len, dtype=np.int64), _i32(blk_weight)
        r = (c_dbl * 2)()
        self.check(lib.fh_vec_wdot(self.h, int(bl.sum()), len(bl), _np_ptr(bl), _np_ptr(bw), c_void_p(x.data_ptr()),
                                   c_void_p(y.data_ptr()), r), "fh_vec_wdot")
        return complex(r[0], r[1])

    def fh_vec_lanczos_update(self, blk_len, blk_weight, a_raw, bj2, bjm2, tol, uj, uprev, w):
        bl, bw = np.ascontiguousarray(blk_len, dtype=np.int64), _i32(blk_weight)
        r = c_dbl()
        self.check(lib.fh_vec_lanczos_update(self.h, int(bl.sum()), len(bl), _np_ptr(bl), _np_ptr(bw), a_raw, bj2, bjm2, tol,
                                             c_void_p(uj.data_ptr()), c_void_p(uprev.data_ptr() if uprev is not None else 0),
                                             c_void_p(w.data_ptr()), C.byref(r)), "fh_vec_lanczos_update")
        return r.value

    def fh_zgemm_split(self, M, N, segs, conj_a, A, B, C, ldc):
        """segs: list of (K, alpha, a_off, a_sm, a_sk, b_off, b_sk, b_sn); A, B, C complex128 CUDA tensors."""
        K, sm_, sk_, bk_, bn_ = (_i32([g[i] for g in segs]) for i in (0, 3, 4, 6, 7))
        al = np.ascontiguousarray([g[1] for g in segs], dtype=np.float64)
        ao, bo = (np.ascontiguousarray([g[i] for g in segs], dtype=np.int64) for i in (2, 5))
        self.check(lib.fh_zgemm_split(self.h, M, N, len(segs), _np_ptr(K), _np_ptr(al), int(conj_a), c_void_p(A.data_ptr()),
                                      _np_ptr(ao), _np_ptr(sm_), _np_ptr(sk_), c_void_p(B.data_ptr()), _np_ptr(bo),
                                      _np_ptr(bk_), _np_ptr(bn_), c_void_p(C.data_ptr()), ldc), "fh_zgemm_split")

    def fh_vec_lincomb(self, coef, V, stride, y):
        c = np.ascontiguousarray(coef, dtype=np.complex128)
        self.check(lib.fh_vec_lincomb(self.h, int(y.numel()), len(c), _np_ptr(c), c_void_p(V.data_ptr()), int(stride),
                                      c_void_p(y.data_ptr())), "fh_vec_lincomb")

    def fh_copy_blocks(self, src_off, dst_off, rows, cols, ld_src, ld_dst, transpose, scale, src, dst):
        so, do = np.ascontiguousarray(src_off, dtype=np.int64), np.ascontiguousarray(dst_off, dtype=np.int64)
        sc = np.ascontiguousarray(scale, dtype=np.float64)
        arrs = [_i32(a) for a in (rows, cols, ld_src, ld_dst, transpose)]
        self.check(lib.fh_copy_blocks(self.h, len(so), _np_ptr(so), _np_ptr(do), *[_np_ptr(a) for a in arrs], _np_ptr(sc),
                                      c_void_p(src.data_ptr()), c_void_p(dst.data_ptr())), "fh_copy_blocks")

    def heff_flops(self):
        return int(lib.heff_flops(self.h))

    def heff_inner(self, x, y):
        r = (c_dbl * 2)()
        self.check(lib.heff_inner(self.h, c_void_p(x.data_ptr()), c_void_p(y.data_ptr()), r), "heff_inner")
        return complex(r[0], r[1])

    def heff_expm(self, theta, out, tau, krylov_dim):
        self.check(lib.heff_expm(self.h, c_void_p(theta.data_ptr()), c_void_p(out.data_ptr()), tau, krylov_dim), "heff_expm")

    def heff_expm_adaptive(self, theta, out, tau, krylov_dim, adapt_tol):
        k = c_int(0)
        self.check(lib.heff_expm_adaptive(self.h, c_void_p(theta.data_ptr()), c_void_p(out.data_ptr()), tau,
                                          krylov_dim, adapt_tol, C.byref(k)), "heff_expm_adaptive")
        return k.value

    def fh_factorization_stats(self):
        a = (C.c_int64 * 9)()
        self.check(lib.fh_factorization_stats(self.h, a), "fh_factorization_stats")
        return dict(jacobi_kernel=a[0], gesvdp=a[1], gesvd=a[2], gesvdp_rejected=a[3], qr=a[4], qr_kernel=a[5],
                    jacobi_mid_kernel=a[6], gram_eig=a[7], gram_redone=a[8])

    def fh_get_traffic(self):
        a, b = c_i64(0), c_i64(0)
        self.check(lib.fh_get_traffic(self.h, C.byref(a), C.byref(b)), "fh_get_traffic")
        return dict(vec_bytes=a.value, pack_bytes=b.value)

    def fh_enable_timers(self, on):
        self.check(lib.fh_enable_timers(self.h, 1 if on else 0), "fh_enable_timers")

    def fh_plan_cache_stats(self, mps):
        a, b, c = C.c_int64(0), C.c_int64(0), C.c_int64(0)
        self.check(lib.fh_plan_cache_stats(mps, C.byref(a), C.byref(b), C.byref(c)), "fh_plan_cache_stats")
        return dict(hits=a.value, misses=b.value, host_bytes=c.value)

    def fh_plan_cache_limit(self, mps, max_host_bytes):
        self.check(lib.fh_plan_cache_limit(mps, int(max_host_bytes)), "fh_plan_cache_limit")

    def fh_krylov_stats(self):
        a, b = C.c_int64(0), C.c_int64(0)
        self.check(lib.fh_krylov_stats(self.h, C.byref(a), C.byref(b)), "fh_krylov_stats")
        return a.value, b.value

    def tdvp2_sweep(self, mpo, mps, dt, krylov_dim=10, krylov_tol=1e-12, chi_max_full=1 << 30, eps_trunc=-1.0,
                    krylov_adapt_tol=0.0):
        p = fh_params(krylov_dim, krylov_tol, chi_max_full, eps_trunc, krylov_adapt_tol)
        self.check(lib.tdvp2_sweep(self.h, mpo, mps, dt, C.byref(p)), "tdvp2_sweep")

    def tdvp_sweep_auto(self, mpo, mps, dt, krylov_dim=10, krylov_tol=1e-12, chi_max_full=1 << 30, eps_trunc=-1.0,
                        krylov_adapt_tol=0.0):
        p = fh_params(krylov_dim, krylov_tol, chi_max_full, eps_trunc, krylov_adapt_tol)
        n = c_int(0)
        self.check(lib.tdvp_sweep_auto(self.h, mpo, mps, dt, C.byref(p), C.byref(n)), "tdvp_sweep_auto")
        return n.value

    def tdvp1_sweep(self, mpo, mps, dt, krylov_dim=10, krylov_tol=1e-12, krylov_adapt_tol=0.0):
        p = fh_params(krylov_dim, krylov_tol, 1 << 30, -1.0, krylov_adapt_tol)
        self.check(lib.tdvp1_sweep(self.h, mpo, mps, dt, C.byref(p)), "tdvp1_sweep")

    def tdvp2_last_stats(self):
        d, a, b, c = c_dbl(), c_int(), c_int(), c_int()
        self.check(lib.tdvp2_last_stats(self.h, C.byref(d), C.byref(a), C.byref(b), C.byref(c)), "tdvp2_last_stats")
        return dict(max_discarded=d.value, chi_full=a.value, chi_su2=b.value, dmax=c.value)

    def measure_local(self, mps, L):
        n, sz, dc = np.zeros(L), np.zeros(L), np.zeros(L)
        self.check(lib.measure_local(self.h, mps, _np_ptr(n), _np_ptr(sz), _np_ptr(dc)), "measure_local")
        return dict(n=n, sz=sz, docc=dc)

    def measure_global(self, mpo, mps):
        a, b = c_dbl(), c_dbl()
        self.check(lib.measure_global(self.h, mpo, mps, C.byref(a), C.byref(b)), "measure_global")
        return dict(norm2=a.value, energy=b.value)

    def fh_get_timers(self):
        v = [c_dbl() for _ in range(5)]
        self.check(lib.fh_get_timers(self.h, *[C.byref(x) for x in v]), "fh_get_timers")
        return dict(zip(("heff", "env", "svd", "vec", "pack"), [x.value for x in v]))

    def fh_reset_timers(self):
        self.check(lib.fh_reset_timers(self.h), "fh_reset_timers")

    def fh_launch_count(self):
        return int(lib.fh_launch_count(self.h))

    OPT_GEMM_PATH, OPT_SVD_MID_MAXN, OPT_SVD_THREADS, OPT_SVD_SMALL_MAXN, OPT_SYMMETRY, OPT_PRECISION, OPT_SVD_GRAM_MINN, OPT_SVD_GRAM_BATCH_MAXN = 1, 2, 3, 4, 5, 6, 7, 8

    def fh_set_option(self, key, value):
        self.check(lib.fh_set_option(self.h, int(key), int(value)), "fh_set_option")

    def fh_arena_stats(self):
        a, b = c_size_t(), c_size_t()
        self.check(lib.fh_arena_stats(self.h, C.byref(a), C.byref(b)), "fh_arena_stats")
        return a.value, b.value

    def fh_cublas_gemm_seconds(self, n, is_complex, reps):
        s = c_dbl()
        self.check(lib.fh_cublas_gemm_seconds(self.h, n, int(is_complex), reps, C.byref(s)), "fh_cublas_gemm_seconds")
        return s.value
