"""Thin ctypes binding over libschwarmax.so (include/schwarmax.h): argument marshalling only.

Every step of the path runs in the CUDA kernels; torch supplies device memory and streams.  There is
no CPU fallback: if the library is missing or no CUDA device is present the calls raise.
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
SO = os.path.join(HERE, "libschwarmax.so")
SM_F64, SM_F32 = 0, 1
PRECISION = {"f64": SM_F64, "f32": SM_F32, SM_F64: SM_F64, SM_F32: SM_F32}
EXPORTS = ["sm_make_potential", "sm_make_potential_batch", "sm_free_potential", "sm_build_library",
           "sm_build_library_batch", "sm_build_bundled_library", "sm_build_observable_library", "sm_build_gh_library", "sm_build_observable_library_batch", "sm_build_gh_library_batch", "sm_stage_library_batch", "sm_stage_library_noalloc", "sm_flush_rows", "sm_scatter_rows", "sm_flush_rows_compact", "sm_zero_async", "sm_solve_weights", "sm_marginal_chi2", "sm_debug_gemm_f64", "sm_debug_invert_spd", "sm_eval_force", "sm_integrate_trajectories", "sm_integrate_rk32", "sm_build_library_rk32", "sm_build_observable_library_rk32", "sm_build_gh_library_rk32", "sm_build_observable_library_rk32_batch", "sm_build_gh_library_rk32_batch", "sm_set_debug_flags",
           "sm_measure_fma_peak", "sm_last_kernel_times", "sm_last_solve_times", "sm_launch_count", "sm_last_error", "sm_version", "sm_debug_host_force", "sm_debug_host_lambda"]


class SmComponent(C.Structure):
    _fields_ = [("kind", C.c_int), ("rotating", C.c_int), ("p", C.c_double * 6)]


class SmPotentialDesc(C.Structure):
    _fields_ = [("G", C.c_double), ("omega_p", C.c_double), ("phase0", C.c_double),
                ("n_comp", C.c_int), ("comp", SmComponent * 8)]


class SmProjection(C.Structure):
    _fields_ = [("alpha", C.c_double), ("beta", C.c_double), ("gamma", C.c_double)]


class SmGrids(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nv", C.c_int),
                ("x0", C.c_double), ("x1", C.c_double), ("y0", C.c_double), ("y1", C.c_double),
                ("v0", C.c_double), ("v1", C.c_double),
                ("dx", C.c_int), ("dy", C.c_int), ("dz", C.c_int),
                ("bx0", C.c_double), ("bx1", C.c_double), ("by0", C.c_double), ("by1", C.c_double),
                ("bz0", C.c_double), ("bz1", C.c_double)]


class SchwarmaxError(RuntimeError):
    pass


_lib = None


def lib():
    """Load the CUDA extension; fails loudly when it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(SO):
            raise SchwarmaxError(f"{SO} is missing: run `python -m paper_2607_00117_b200.build` "
                                 "(there is no CPU fallback)")
        _lib = C.CDLL(SO)
        _lib.sm_last_error.restype = C.c_char_p
        _lib.sm_launch_count.restype = C.c_int64
        _lib.sm_free_potential.restype = None
    return _lib


def _check(rc, what):
    if rc != 0:
        raise SchwarmaxError(f"{what} failed ({rc}): {lib().sm_last_error().decode()}")


def _desc(spec):
    d = SmPotentialDesc()
    d.G, d.omega_p, d.phase0 = spec["G"], spec.get("omega_p", 0.0), spec.get("phase0", 0.0)
    comps = spec["components"]
    d.n_comp = len(comps)
    if len(comps) > 8:
        raise SchwarmaxError("at most 8 components")
    for i, (kind, rot, p) in enumerate(comps):
        d.comp[i].kind, d.comp[i].rotating = int(kind), int(rot)
        for j, v in enumerate(p):
            d.comp[i].p[j] = float(v)
    return d


def _grids(g):
    out = SmGrids()
    for k, v in g.items():
        setattr(out, k, v)
    return out


def _stream(stream):
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else None


class Potential:
    """Opaque sm_potential handle (one or many trials)."""

    def __init__(self, specs):
        self.specs = list(specs)
        self.n_trials = len(self.specs)
        arr = (SmPotentialDesc * self.n_trials)(*[_desc(s) for s in self.specs])
        self._h = C.c_void_p()
        _check(lib().sm_make_potential_batch(arr, C.c_int(self.n_trials), C.byref(self._h)), "sm_make_potential")

    def close(self):
        if getattr(self, "_h", None):
            lib().sm_free_potential(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def sm_make_potential(spec):
    return Potential([spec])


def sm_make_potential_batch(specs):
    return Potential(specs)


def sm_free_potential(pot):
    pot.close()


def _dev_f64(x):
    import torch
    if isinstance(x, torch.Tensor):
        if not x.is_cuda or x.dtype != torch.float64 or not x.is_contiguous():
            raise SchwarmaxError("expected a contiguous float64 CUDA tensor")
        return x
    return torch.as_tensor(np.ascontiguousarray(x, dtype=np.float64)).cuda()


def sm_build_library(pot, ics, dt, n_steps, stride, projections, grids, precision="f64", losvd=None, dens=None,
                     nout=None, want_nout=True, want_diag=False, stream=None):
    """-> dict(losvd[n_proj,n_orb,nlos] f32, dens[n_orb,nden] f32, nout[n_proj+1,n_orb] i32, diag[n_orb,2] f64)."""
    import torch
    ics = _dev_f64(ics)
    n_orb = ics.shape[0]
    g = _grids(grids)
    nlos, nden, n_proj = g.nx * g.ny * g.nv, g.dx * g.dy * g.dz, len(projections)
    P = (SmProjection * n_proj)(*[SmProjection(*p) for p in projections])
    dev = ics.device
    if losvd is None:
        losvd = torch.empty((n_proj, n_orb, nlos), dtype=torch.float32, device=dev)
    if dens is None:
        dens = torch.empty((n_orb, nden), dtype=torch.float32, device=dev)
    if nout is None and want_nout:
        nout = torch.empty((n_proj + 1, n_orb), dtype=torch.int32, device=dev)
    diag = torch.empty((n_orb, 2), dtype=torch.float64, device=dev) if want_diag else None
    _check(lib().sm_build_library(pot._h, _ptr(ics), C.c_int64(n_orb), C.c_double(dt), C.c_int64(n_steps),
                                  C.c_int32(stride), P, C.c_int(n_proj), C.byref(g), C.c_int(PRECISION[precision]),
                                  _ptr(losvd), _ptr(dens), _ptr(nout), _ptr(diag), _stream(stream)), "sm_build_library")
    return {"losvd": losvd, "dens": dens, "nout": nout, "diag": diag}


def sm_build_library_batch(pot, ics, dt, n_steps, stride, projections, grids, precision="f32", trial0=0, n_trials=None,
                           losvd=None, dens=None, nout=None, want_nout=True, stream=None):
    """ics: [n_orb,6] shared or [n_trials,n_orb,6]; projections: [n_trials][n_proj] of (alpha,beta,gamma)."""
    import torch
    ics = _dev_f64(ics)
    n_trials = pot.n_trials - trial0 if n_trials is None else n_trials
    per_trial = ics.dim() == 3
    n_orb = ics.shape[-2]
    if per_trial and ics.shape[0] != n_trials:
        raise SchwarmaxError("ics leading dimension must equal n_trials")
    g = _grids(grids)
    nlos, nden, n_proj = g.nx * g.ny * g.nv, g.dx * g.dy * g.dz, len(projections[0])
    flat = [SmProjection(*p) for tr in projections for p in tr]
    if len(flat) != n_trials * n_proj:
        raise SchwarmaxError("projections must be [n_trials][n_proj]")
    P = (SmProjection * len(flat))(*flat)
    dev = ics.device
    if losvd is None:
        losvd = torch.empty((n_trials, n_proj, n_orb, nlos), dtype=torch.float32, device=dev)
    if dens is None:
        dens = torch.empty((n_trials, n_orb, nden), dtype=torch.float32, device=dev)
    if nout is None and want_nout:
        nout = torch.empty((n_trials, n_proj + 1, n_orb), dtype=torch.int32, device=dev)
    _check(lib().sm_build_library_batch(pot._h, C.c_int(trial0), C.c_int(n_trials), _ptr(ics), C.c_int(int(per_trial)),
                                        C.c_int64(n_orb), C.c_double(dt), C.c_int64(n_steps), C.c_int32(stride), P,
                                        C.c_int(n_proj), C.byref(g), C.c_int(PRECISION[precision]), _ptr(losvd),
                                        _ptr(dens), _ptr(nout), _stream(stream)), "sm_build_library_batch")
    return {"losvd": losvd, "dens": dens, "nout": nout}


def sm_build_bundled_library(pot, ics, dt, n_steps, stride, projections, grids, n_bundle=1, fourfold=True, precision="f64",
                             losvd=None, dens=None, nout=None, want_nout=True, stream=None):
    """Symmetrised orbit bundles -> dict(losvd[n_proj,n_rows,nlos], dens[n_rows,nden], nout[n_proj+1,n_rows]), n_rows = n_orb/n_bundle."""
    import torch
    ics = _dev_f64(ics)
    n_orb = ics.shape[0]
    n_rows = n_orb // n_bundle
    g = _grids(grids)
    nlos, nden, n_proj = g.nx * g.ny * g.nv, g.dx * g.dy * g.dz, len(projections)
    P = (SmProjection * n_proj)(*[SmProjection(*p) for p in projections])
    dev = ics.device
    if losvd is None:
        losvd = torch.empty((n_proj, n_rows, nlos), dtype=torch.float32, device=dev)
    if dens is None:
        dens = torch.empty((n_rows, nden), dtype=torch.float32, device=dev)
    if nout is None and want_nout:
        nout = torch.empty((n_proj + 1, n_rows), dtype=torch.int32, device=dev)
    _check(lib().sm_build_bundled_library(pot._h, _ptr(ics), C.c_int64(n_orb), C.c_double(dt), C.c_int64(n_steps),
                                          C.c_int32(stride), P, C.c_int(n_proj), C.byref(g), C.c_int(PRECISION[precision]),
                                          C.c_int32(n_bundle), C.c_int(int(fourfold)), _ptr(losvd), _ptr(dens), _ptr(nout),
                                          _stream(stream)), "sm_build_bundled_library")
    return {"losvd": losvd, "dens": dens, "nout": nout}


def sm_build_observable_library(pot, ics, dt, n_steps, stride, projections, grids, ap_map, n_ap, n_bundle=1, fourfold=False,
                                precision="f64", density_mode=0, losvd=None, dens=None, nout=None, stream=None):
    """Aperture-regrouped rows -> dict(losvd[n_proj,n_rows,n_ap*nv], dens[n_rows,nden], nout[n_proj+1,n_rows]);
    ap_map: int32 [ny*nx] (numpy or CUDA tensor), < 0 = pixel without aperture, None = plain pixels;
    density_mode 1 = cylindrical (R, phi, z) density cells."""
    import torch
    ics = _dev_f64(ics)
    n_orb = ics.shape[0]
    n_rows = n_orb // n_bundle
    g = _grids(grids)
    if ap_map is not None and not isinstance(ap_map, torch.Tensor):
        ap_map = torch.as_tensor(np.ascontiguousarray(ap_map, dtype=np.int32)).cuda()
    if ap_map is not None and (ap_map.dtype != torch.int32 or not ap_map.is_cuda or ap_map.numel() != g.nx * g.ny
                               or not ap_map.is_contiguous()):
        raise SchwarmaxError("ap_map must be a contiguous int32 CUDA tensor with ny*nx entries")
    nlos, nden, n_proj = (n_ap if ap_map is not None else g.nx * g.ny) * g.nv, g.dx * g.dy * g.dz, len(projections)
    P = (SmProjection * n_proj)(*[SmProjection(*p) for p in projections])
    dev = ics.device
    if losvd is None:
        losvd = torch.empty((n_proj, n_rows, nlos), dtype=torch.float32, device=dev)
    if dens is None:
        dens = torch.empty((n_rows, nden), dtype=torch.float32, device=dev)
    if nout is None:
        nout = torch.empty((n_proj + 1, n_rows), dtype=torch.int32, device=dev)
    _check(lib().sm_build_observable_library(pot._h, _ptr(ics), C.c_int64(n_orb), C.c_double(dt), C.c_int64(n_steps),
                                             C.c_int32(stride), P, C.c_int(n_proj), C.byref(g), C.c_int(PRECISION[precision]),
                                             C.c_int32(n_bundle), C.c_int(int(fourfold)), _ptr(ap_map), C.c_int32(n_ap),
                                             C.c_int(density_mode), _ptr(losvd), _ptr(dens), _ptr(nout), _stream(stream)), "sm_build_observable_library")
    return {"losvd": losvd, "dens": dens, "nout": nout}


def sm_build_gh_library(pot, ics, dt, n_steps, stride, projections, grids, ap_map, n_ap, v0, s, n_bundle=1, fourfold=False,
                        precision="f64", density_mode=0, gh=None, dens=None, nout=None, stream=None):
    """Gauss-Hermite matrices -> dict(gh[n_proj,n_rows,n_ap,6] f32, dens[n_rows,nden] f32, nout[n_proj+1,n_rows] i32)."""
    import torch
    ics = _dev_f64(ics)
    n_orb = ics.shape[0]
    n_rows = n_orb // n_bundle
    g = _grids(grids)
    if not isinstance(ap_map, torch.Tensor):
        ap_map = torch.as_tensor(np.ascontiguousarray(ap_map, dtype=np.int32)).cuda()
    v0, s = _dev_f64(v0), _dev_f64(s)
    if ap_map.dtype != torch.int32 or ap_map.numel() != g.nx * g.ny or v0.numel() != n_ap or s.numel() != n_ap:
        raise SchwarmaxError("ap_map must be int32 with ny*nx entries; v0 and s need n_ap entries")
    nden, n_proj = g.dx * g.dy * g.dz, len(projections)
    P = (SmProjection * n_proj)(*[SmProjection(*p) for p in projections])
    dev = ics.device
    if gh is None:
        gh = torch.empty((n_proj, n_rows, n_ap, 6), dtype=torch.float32, device=dev)
    if dens is None:
        dens = torch.empty((n_rows, nden), dtype=torch.float32, device=dev)
    if nout is None:
        nout = torch.empty((n_proj + 1, n_rows), dtype=torch.int32, device=dev)
    _check(lib().sm_build_gh_library(pot._h, _ptr(ics), C.c_int64(n_orb), C.c_double(dt), C.c_int64(n_steps), C.c_int32(stride),
                                     P, C.c_int(n_proj), C.byref(g), C.c_int(PRECISION[precision]), C.c_int32(n_bundle),
                                     C.c_int(int(fourfold)), _ptr(ap_map), C.c_int32(n_ap), _ptr(v0), _ptr(s),
                                     C.c_int(density_mode), _ptr(gh), _ptr(dens), _ptr(nout), _stream(stream)), "sm_build_gh_library")
    return {"gh": gh, "dens": dens, "nout": nout}


def sm_build_observable_library_batch(pot, ics, dt, n_steps, stride, projections, grids, ap_map=None, n_ap=0, n_bundle=1,
                                      fourfold=False, precision="f64", density_mode=0, gh=None, trial0=0, n_trials=None,
                                      out=None, stream=None):
    """The bundled / aperture / cylindrical / Gauss-Hermite row forms for a range of trials in one integrator launch.
    ics: [n_orb,6] shared or [n_trials,n_orb,6]; projections: [n_trials][n_proj]; gh = (v0[n_ap], s[n_ap]) switches to
    Gauss-Hermite rows.  -> dict(losvd[n_trials,n_proj,n_rows,cells] or gh[n_trials,n_proj,n_rows,n_ap,6],
    dens[n_trials,n_rows,nden], nout[n_trials,n_proj+1,n_rows])."""
    import torch
    ics = _dev_f64(ics)
    n_trials = pot.n_trials - trial0 if n_trials is None else n_trials
    per_trial = ics.dim() == 3
    n_orb = ics.shape[-2]
    n_rows = n_orb // max(n_bundle, 1)
    g = _grids(grids)
    n_proj = len(projections[0])
    flat = [SmProjection(*p) for tr in projections for p in tr]
    if len(flat) != n_trials * n_proj:
        raise SchwarmaxError("projections must be [n_trials][n_proj]")
    P = (SmProjection * len(flat))(*flat)
    dev = ics.device
    if ap_map is not None and not isinstance(ap_map, torch.Tensor):
        ap_map = torch.as_tensor(np.ascontiguousarray(ap_map, dtype=np.int32)).to(dev)
    if ap_map is not None and (ap_map.dtype != torch.int32 or not ap_map.is_cuda or ap_map.numel() != g.nx * g.ny or not ap_map.is_contiguous()):
        raise SchwarmaxError("ap_map must be a contiguous int32 CUDA tensor with ny*nx entries")
    nden = g.dx * g.dy * g.dz
    if out is None:
        out = dict(dens=torch.empty((n_trials, n_rows, nden), dtype=torch.float32, device=dev),
                   nout=torch.empty((n_trials, n_proj + 1, n_rows), dtype=torch.int32, device=dev))
        if gh is not None:
            out["gh"] = torch.empty((n_trials, n_proj, n_rows, n_ap, 6), dtype=torch.float32, device=dev)
        else:
            out["losvd"] = torch.empty((n_trials, n_proj, n_rows, (n_ap if ap_map is not None else g.nx * g.ny) * g.nv), dtype=torch.float32, device=dev)
    head = (pot._h, C.c_int(trial0), C.c_int(n_trials), _ptr(ics), C.c_int(int(per_trial)), C.c_int64(n_orb), C.c_double(dt),
            C.c_int64(n_steps), C.c_int32(stride), P, C.c_int(n_proj), C.byref(g), C.c_int(PRECISION[precision]), C.c_int32(n_bundle),
            C.c_int(int(fourfold)), _ptr(ap_map), C.c_int32(n_ap))
    if gh is not None:
        v0, s = _dev_f64(gh[0]), _dev_f64(gh[1])
        if ap_map is None or v0.numel() != n_ap or s.numel() != n_ap:
            raise SchwarmaxError("Gauss-Hermite rows need an aperture map and n_ap entries of v0 and s")
        _check(lib().sm_build_gh_library_batch(*head, _ptr(v0), _ptr(s), C.c_int(density_mode), _ptr(out["gh"]), _ptr(out["dens"]),
                                               _ptr(out["nout"]), _stream(stream)), "sm_build_gh_library_batch")
    else:
        _check(lib().sm_build_observable_library_batch(*head, C.c_int(density_mode), _ptr(out["losvd"]), _ptr(out["dens"]),
                                                       _ptr(out["nout"]), _stream(stream)), "sm_build_observable_library_batch")
    return out


def sm_stage_library_batch(pot, ics, dt, n_steps, stride, projections, grids, precision="f64", trial0=0, n_trials=None,
                           stage=None, stream=None):
    """-> stage[n_trials, n_proj+1, n_orb, n_rec] uint32 cell indices (int32 tensor, -1 = outside the grid).
    ics: [n_orb,6] shared or [n_trials,n_orb,6]; projections: [n_trials][n_proj]."""
    import torch
    ics = _dev_f64(ics)
    n_trials = pot.n_trials - trial0 if n_trials is None else n_trials
    per_trial = ics.dim() == 3
    n_orb = ics.shape[-2]
    g = _grids(grids)
    n_proj = len(projections[0])
    flat = [SmProjection(*p) for tr in projections for p in tr]
    if len(flat) != n_trials * n_proj:
        raise SchwarmaxError("projections must be [n_trials][n_proj]")
    P = (SmProjection * len(flat))(*flat)
    n_rec = n_steps // stride
    if stage is None:
        stage = torch.empty((n_trials, n_proj + 1, n_orb, n_rec), dtype=torch.int32, device=ics.device)
    _check(lib().sm_stage_library_batch(pot._h, C.c_int(trial0), C.c_int(n_trials), _ptr(ics), C.c_int(int(per_trial)),
                                        C.c_int64(n_orb), C.c_double(dt), C.c_int64(n_steps), C.c_int32(stride), P,
                                        C.c_int(n_proj), C.byref(g), C.c_int(PRECISION[precision]), _ptr(stage),
                                        _stream(stream)), "sm_stage_library_batch")
    return stage


def sm_stage_library_noalloc(pot, ics, dt, n_steps, stride, projections, grids, precision="f64", trial=0, stage=None, stream=None):
    """sm_stage_library_batch for one trial with all scratch in the library's static device array: allocates nothing
    (pass `stage` to keep torch from allocating either).  -> stage[n_proj+1, n_orb, n_rec] int32, -1 = outside the grid.
    n_orb <= 32768, n_steps <= 65534; calls that overlap on one GPU race (include/schwarmax.h)."""
    import torch
    ics = _dev_f64(ics)
    n_orb = ics.shape[0]
    g = _grids(grids)
    n_proj = len(projections)
    P = (SmProjection * n_proj)(*[SmProjection(*p) for p in projections])
    n_rec = n_steps // stride
    if stage is None:
        stage = torch.empty((n_proj + 1, n_orb, n_rec), dtype=torch.int32, device=ics.device)
    _check(lib().sm_stage_library_noalloc(pot._h, C.c_int(trial), _ptr(ics), C.c_int64(n_orb), C.c_double(dt), C.c_int64(n_steps),
                                          C.c_int32(stride), P, C.c_int(n_proj), C.byref(g), C.c_int(PRECISION[precision]),
                                          _ptr(stage), _stream(stream)), "sm_stage_library_noalloc")
    return stage


def sm_flush_rows(stage, orb0, n_rows, grids, losvd=None, dens=None, nout=None, want_nout=True, stream=None):
    """Dense rows of orbits [orb0, orb0+n_rows) of every trial of stage[n_trials, n_proj+1, n_orb, n_rec]."""
    import torch
    if stage.dim() != 4 or not stage.is_contiguous() or stage.dtype != torch.int32:
        raise SchwarmaxError("stage must be a contiguous int32 tensor [n_trials, n_proj+1, n_orb, n_rec]")
    n_trials, n_hist, n_orb, n_rec = stage.shape
    g = _grids(grids)
    nlos, nden, n_proj = g.nx * g.ny * g.nv, g.dx * g.dy * g.dz, n_hist - 1
    dev = stage.device
    if losvd is None:
        losvd = torch.empty((n_trials, n_proj, n_rows, nlos), dtype=torch.float32, device=dev)
    if dens is None:
        dens = torch.empty((n_trials, n_rows, nden), dtype=torch.float32, device=dev)
    if nout is None and want_nout:
        nout = torch.empty((n_trials, n_hist, n_rows), dtype=torch.int32, device=dev)
    _check(lib().sm_flush_rows(_ptr(stage), C.c_int(n_trials), C.c_int(n_proj), C.c_int64(n_orb), C.c_int64(n_rec),
                               C.c_int64(orb0), C.c_int64(n_rows), C.byref(g), _ptr(losvd), _ptr(dens), _ptr(nout),
                               _stream(stream)), "sm_flush_rows")
    return {"losvd": losvd, "dens": dens, "nout": nout}


def sm_scatter_rows(stage, orb0, n_rows, grids, losvd, dens, nout=None, want_nout=True, stream=None):
    """sm_flush_rows into rows the caller has zeroed (sm_zero_async): only the non-zero cells are written."""
    import torch
    if stage.dim() != 4 or not stage.is_contiguous() or stage.dtype != torch.int32:
        raise SchwarmaxError("stage must be a contiguous int32 tensor [n_trials, n_proj+1, n_orb, n_rec]")
    n_trials, n_hist, n_orb, n_rec = stage.shape
    g = _grids(grids)
    if nout is None and want_nout:
        nout = torch.empty((n_trials, n_hist, n_rows), dtype=torch.int32, device=stage.device)
    _check(lib().sm_scatter_rows(_ptr(stage), C.c_int(n_trials), C.c_int(n_hist - 1), C.c_int64(n_orb), C.c_int64(n_rec),
                                 C.c_int64(orb0), C.c_int64(n_rows), C.byref(g), _ptr(losvd), _ptr(dens), _ptr(nout),
                                 _stream(stream)), "sm_scatter_rows")
    return {"losvd": losvd, "dens": dens, "nout": nout}


def sm_flush_rows_compact(stage, orb0, n_rows, grids, capacity=None, out=None, want_nout=True, stream=None):
    """Rows [orb0, orb0+n_rows) of every trial and histogram of stage[n_trials, n_proj+1, n_orb, n_rec] as (cell, count) pairs.
    -> dict(cell[capacity] i32 (bit pattern of the u32 cell), count[capacity] f32, row_start[n_trials, n_hist, n_rows] i64,
    row_nnz[...] i32, nout[...] i32, total[1] i64).  total > capacity: entries were dropped, call again with a larger capacity."""
    import torch
    if stage.dim() != 4 or not stage.is_contiguous() or stage.dtype != torch.int32:
        raise SchwarmaxError("stage must be a contiguous int32 tensor [n_trials, n_proj+1, n_orb, n_rec]")
    n_trials, n_hist, n_orb, n_rec = stage.shape
    g = _grids(grids)
    dev = stage.device
    if out is None:
        cap = n_trials * n_hist * n_rows * n_rec if capacity is None else capacity
        out = dict(cell=torch.empty(cap, dtype=torch.int32, device=dev), count=torch.empty(cap, dtype=torch.float32, device=dev),
                   row_start=torch.empty((n_trials, n_hist, n_rows), dtype=torch.int64, device=dev),
                   row_nnz=torch.empty((n_trials, n_hist, n_rows), dtype=torch.int32, device=dev),
                   nout=torch.empty((n_trials, n_hist, n_rows), dtype=torch.int32, device=dev) if want_nout else None,
                   total=torch.empty(1, dtype=torch.int64, device=dev))
    cap = out["cell"].numel()
    _check(lib().sm_flush_rows_compact(_ptr(stage), C.c_int(n_trials), C.c_int(n_hist - 1), C.c_int64(n_orb), C.c_int64(n_rec),
                                       C.c_int64(orb0), C.c_int64(n_rows), C.byref(g), C.c_int64(cap), _ptr(out["cell"]),
                                       _ptr(out["count"]), _ptr(out["row_start"]), _ptr(out["row_nnz"]), _ptr(out.get("nout")),
                                       _ptr(out["total"]), _stream(stream)), "sm_flush_rows_compact")
    return out


def sm_zero_async(t, stream=None):
    """Zero a contiguous CUDA tensor on `stream` with the library's small fill kernel (fits beside a running integrator)."""
    if not t.is_contiguous():
        raise SchwarmaxError("expected a contiguous tensor")
    _check(lib().sm_zero_async(_ptr(t), C.c_uint64(t.numel() * t.element_size()), _stream(stream)), "sm_zero_async")
    return t


def sm_eval_force(pot, xyz, t=0.0, precision="f64", trial=0, want_phi=True, stream=None):
    import torch
    xyz = _dev_f64(xyz).reshape(-1, 3)
    F = torch.empty_like(xyz)
    Phi = torch.empty(xyz.shape[0], dtype=torch.float64, device=xyz.device) if want_phi else None
    _check(lib().sm_eval_force(pot._h, C.c_int(trial), _ptr(xyz), C.c_int64(xyz.shape[0]), C.c_double(t),
                               C.c_int(PRECISION[precision]), _ptr(F), _ptr(Phi), _stream(stream)), "sm_eval_force")
    return (F, Phi) if want_phi else F


def sm_integrate_trajectories(pot, ics, dt, n_steps, stride=1, precision="f64", trial=0, stream=None):
    import torch
    ics = _dev_f64(ics)
    n_rec = n_steps // stride
    traj = torch.empty((n_rec, ics.shape[0], 6), dtype=torch.float64, device=ics.device)
    _check(lib().sm_integrate_trajectories(pot._h, C.c_int(trial), _ptr(ics), C.c_int64(ics.shape[0]), C.c_double(dt),
                                           C.c_int64(n_steps), C.c_int32(stride), C.c_int(PRECISION[precision]),
                                           _ptr(traj), _stream(stream)), "sm_integrate_trajectories")
    return traj


def sm_integrate_rk32(pot, ics, n_steps, rtol=1e-4, atol_x=1e-4, atol_v=1e-4, h0=1e-3, stream=None):
    """The paper's adaptive RK3(2) in the rotating frame -> samples [n_steps, n_orb, 6], dt_w [n_steps, n_orb], t_end [n_orb]."""
    import torch
    ics = _dev_f64(ics)
    n = ics.shape[0]
    samples = torch.empty((n_steps, n, 6), dtype=torch.float64, device=ics.device)
    dtw = torch.empty((n_steps, n), dtype=torch.float64, device=ics.device)
    t_end = torch.empty((n,), dtype=torch.float64, device=ics.device)
    _check(lib().sm_integrate_rk32(pot._h, _ptr(ics), C.c_int64(n), C.c_int64(n_steps), C.c_double(rtol), C.c_double(atol_x),
                                   C.c_double(atol_v), C.c_double(h0), _ptr(samples), _ptr(dtw), _ptr(t_end), _stream(stream)),
           "sm_integrate_rk32")
    return samples, dtw, t_end


def sm_build_library_rk32(pot, ics, n_steps, projections, grids, rtol=1e-4, atol_x=1e-4, atol_v=1e-4, h0=1e-3, out=None, stream=None):
    """delta-t-weighted orbit-observable matrices of the adaptive integrator ->
    dict(losvd[n_proj,n_orb,nlos], dens[n_orb,nden], wout[n_proj+1,n_orb], t_end[n_orb]) (fp32 time fractions).
    out: a dict returned by an earlier call of the same shape, overwritten in place (caller-owned buffers)."""
    import torch
    ics = _dev_f64(ics)
    n = ics.shape[0]
    g = _grids(grids)
    nlos, nden = g.nx * g.ny * g.nv, g.dx * g.dy * g.dz
    P = (SmProjection * len(projections))(*[SmProjection(*p) for p in projections])
    if out is not None:
        losvd, dens, wout, t_end = out["losvd"], out["dens"], out["wout"], out["t_end"]
        if tuple(losvd.shape) != (len(projections), n, nlos) or tuple(dens.shape) != (n, nden):
            raise SchwarmaxError("out= buffers have the wrong shape")
    else:
        losvd = torch.empty((len(projections), n, nlos), dtype=torch.float32, device=ics.device)
        dens = torch.empty((n, nden), dtype=torch.float32, device=ics.device)
        wout = torch.empty((len(projections) + 1, n), dtype=torch.float32, device=ics.device)
        t_end = torch.empty((n,), dtype=torch.float64, device=ics.device)
    _check(lib().sm_build_library_rk32(pot._h, _ptr(ics), C.c_int64(n), C.c_int64(n_steps), C.c_double(rtol), C.c_double(atol_x),
                                       C.c_double(atol_v), C.c_double(h0), P, C.c_int(len(projections)), C.byref(g), _ptr(losvd),
                                       _ptr(dens), _ptr(wout), _ptr(t_end), _stream(stream)), "sm_build_library_rk32")
    return dict(losvd=losvd, dens=dens, wout=wout, t_end=t_end)


def sm_build_observable_library_rk32(pot, ics, n_steps, projections, grids, ap_map=None, n_ap=0, n_bundle=1, fourfold=False,
                                     density_mode=0, gh=None, rtol=1e-4, atol_x=1e-4, atol_v=1e-4, h0=1e-3, want_diag=False,
                                     out=None, stream=None):
    """The paper's observables on the adaptive integrator.  gh = (v0[n_ap], s[n_ap]) switches to Gauss-Hermite rows
    (sm_build_gh_library_rk32).  -> dict(losvd[n_proj,n_rows,n_cells] or gh[n_proj,n_rows,n_ap,6], dens, wout[n_proj+1,n_rows],
    t_end[n_orb], diag[n_orb,2] or None)."""
    import torch
    ics = _dev_f64(ics)
    n_orb = ics.shape[0]
    g = _grids(grids)
    n_proj = len(projections)
    P = (SmProjection * n_proj)(*[SmProjection(*p) for p in projections])
    dev = ics.device
    n_rows = n_orb // max(n_bundle, 1)
    if ap_map is not None and not isinstance(ap_map, torch.Tensor):
        ap_map = torch.as_tensor(np.ascontiguousarray(ap_map, dtype=np.int32)).to(dev)
    n_cells = (n_ap if ap_map is not None else g.nx * g.ny) * g.nv
    if out is None:
        out = dict(dens=torch.empty((n_rows, g.dx * g.dy * g.dz), dtype=torch.float32, device=dev),
                   wout=torch.empty((n_proj + 1, n_rows), dtype=torch.float32, device=dev),
                   t_end=torch.empty(n_orb, dtype=torch.float64, device=dev),
                   diag=torch.empty((n_orb, 2), dtype=torch.float64, device=dev) if want_diag else None)
        if gh is not None:
            out["gh"] = torch.empty((n_proj, n_rows, n_ap, 6), dtype=torch.float32, device=dev)
        else:
            out["losvd"] = torch.empty((n_proj, n_rows, n_cells), dtype=torch.float32, device=dev)
    common = (pot._h, _ptr(ics), C.c_int64(n_orb), C.c_int64(n_steps), C.c_double(rtol), C.c_double(atol_x), C.c_double(atol_v),
              C.c_double(h0), P, C.c_int(n_proj), C.byref(g), C.c_int32(n_bundle), C.c_int(int(fourfold)), _ptr(ap_map), C.c_int32(n_ap))
    if gh is not None:
        v0, s = _dev_f64(gh[0]), _dev_f64(gh[1])
        _check(lib().sm_build_gh_library_rk32(*common, _ptr(v0), _ptr(s), C.c_int(density_mode), _ptr(out["gh"]), _ptr(out["dens"]),
                                              _ptr(out["wout"]), _ptr(out["t_end"]), _ptr(out.get("diag")), _stream(stream)),
               "sm_build_gh_library_rk32")
    else:
        _check(lib().sm_build_observable_library_rk32(*common, C.c_int(density_mode), _ptr(out["losvd"]), _ptr(out["dens"]),
                                                      _ptr(out["wout"]), _ptr(out["t_end"]), _ptr(out.get("diag")), _stream(stream)),
               "sm_build_observable_library_rk32")
    return out


def sm_build_observable_library_rk32_batch(pot, ics, n_steps, projections, grids, ap_map=None, n_ap=0, n_bundle=1, fourfold=False,
                                           density_mode=0, gh=None, rtol=1e-4, atol_x=1e-4, atol_v=1e-4, h0=1e-3, want_diag=False,
                                           trial0=0, n_trials=None, out=None, stream=None):
    """The paper's observables on the adaptive integrator for a range of trial potentials in one launch per orbit chunk.
    ics: [n_orb,6] shared or [n_trials,n_orb,6]; projections [n_trials][n_proj]; gh = (v0, s) switches to Gauss-Hermite rows.
    -> dict(losvd[n_trials,n_proj,n_rows,cells] or gh[n_trials,n_proj,n_rows,n_ap,6], dens[n_trials,n_rows,nden],
    wout[n_trials,n_proj+1,n_rows], t_end[n_trials,n_orb], diag[n_trials,n_orb,2] or None)."""
    import torch
    ics = _dev_f64(ics)
    n_trials = pot.n_trials - trial0 if n_trials is None else n_trials
    per_trial = ics.dim() == 3
    n_orb = ics.shape[-2]
    g = _grids(grids)
    n_proj = len(projections[0])
    flat = [SmProjection(*p) for tr in projections for p in tr]
    if len(flat) != n_trials * n_proj:
        raise SchwarmaxError("projections must be [n_trials][n_proj]")
    P = (SmProjection * len(flat))(*flat)
    dev = ics.device
    n_rows = n_orb // max(n_bundle, 1)
    if ap_map is not None and not isinstance(ap_map, torch.Tensor):
        ap_map = torch.as_tensor(np.ascontiguousarray(ap_map, dtype=np.int32)).to(dev)
    n_cells = (n_ap if ap_map is not None else g.nx * g.ny) * g.nv
    if out is None:
        out = dict(dens=torch.empty((n_trials, n_rows, g.dx * g.dy * g.dz), dtype=torch.float32, device=dev),
                   wout=torch.empty((n_trials, n_proj + 1, n_rows), dtype=torch.float32, device=dev),
                   t_end=torch.empty((n_trials, n_orb), dtype=torch.float64, device=dev),
                   diag=torch.empty((n_trials, n_orb, 2), dtype=torch.float64, device=dev) if want_diag else None)
        if gh is not None:
            out["gh"] = torch.empty((n_trials, n_proj, n_rows, n_ap, 6), dtype=torch.float32, device=dev)
        else:
            out["losvd"] = torch.empty((n_trials, n_proj, n_rows, n_cells), dtype=torch.float32, device=dev)
    common = (pot._h, C.c_int(trial0), C.c_int(n_trials), _ptr(ics), C.c_int(int(per_trial)), C.c_int64(n_orb), C.c_int64(n_steps),
              C.c_double(rtol), C.c_double(atol_x), C.c_double(atol_v), C.c_double(h0), P, C.c_int(n_proj), C.byref(g), C.c_int32(n_bundle),
              C.c_int(int(fourfold)), _ptr(ap_map), C.c_int32(n_ap))
    if gh is not None:
        v0, s = _dev_f64(gh[0]), _dev_f64(gh[1])
        _check(lib().sm_build_gh_library_rk32_batch(*common, _ptr(v0), _ptr(s), C.c_int(density_mode), _ptr(out["gh"]), _ptr(out["dens"]),
                                                    _ptr(out["wout"]), _ptr(out["t_end"]), _ptr(out.get("diag")), _stream(stream)),
               "sm_build_gh_library_rk32_batch")
    else:
        _check(lib().sm_build_observable_library_rk32_batch(*common, C.c_int(density_mode), _ptr(out["losvd"]), _ptr(out["dens"]),
                                                            _ptr(out["wout"]), _ptr(out["t_end"]), _ptr(out.get("diag")), _stream(stream)),
               "sm_build_observable_library_rk32_batch")
    return out


class SmWeightBlock(C.Structure):
    _fields_ = [("d_rows", C.c_void_p), ("row_pitch", C.c_int64), ("col0", C.c_int32), ("col_stride", C.c_int32),
                ("n_cols", C.c_int32)]


def sm_solve_weights(blocks, target, sigma, lam, rho, n_iter, xi=None, keep=None, wtilde=None, want_resid=True, want_chi2=False,
                     stream=None):
    """ADMM NNLS for the orbital weights.

    want_chi2 adds chi2 [n_rhs][n_blocks] (Eq. 5 terms against the unperturbed data).
    blocks: list of (matrix, col0, col_stride, n_cols) with matrix a CUDA float32 tensor whose first axis is the orbit
    (row) axis and whose remaining axes are contiguous; (matrix,) alone takes every column.  target, sigma [n_con],
    xi [n_rhs][n_con] or None (one unperturbed right-hand side).  -> dict(w[n_rhs,n_orb] f64, resid[n_rhs,2] f64)."""
    import torch
    arr = (SmWeightBlock * len(blocks))()
    n_orb, n_con, hold = None, 0, []
    for k, blk in enumerate(blocks):
        m = blk[0]
        if m.dtype != torch.float32 or not m.is_cuda or not m.is_contiguous():
            raise SchwarmaxError("weight blocks must be contiguous CUDA float32 tensors")
        pitch = m[0].numel()
        col0, stride, n_cols = (0, 1, pitch) if len(blk) == 1 else blk[1:]
        if n_orb is None:
            n_orb = m.shape[0]
        if m.shape[0] != n_orb:
            raise SchwarmaxError("weight blocks disagree on the number of rows")
        arr[k] = SmWeightBlock(m.data_ptr(), pitch, col0, stride, n_cols)
        n_con += n_cols
        hold.append(m)
    target, sigma = _dev_f64(target), _dev_f64(sigma)
    if target.numel() != n_con or sigma.numel() != n_con:
        raise SchwarmaxError("target and sigma need n_con entries")
    n_rhs = 1
    if xi is not None:
        xi = _dev_f64(xi).reshape(-1, n_con)
        n_rhs = xi.shape[0]
    if keep is not None:
        keep = torch.as_tensor(keep).to(device=target.device, dtype=torch.uint8).contiguous()
    if wtilde is not None:
        wtilde = _dev_f64(wtilde)
    w = torch.empty((n_rhs, n_orb), dtype=torch.float64, device=target.device)
    resid = torch.empty((n_rhs, 2), dtype=torch.float64, device=target.device) if want_resid else None
    chi2 = torch.empty((n_rhs, len(blocks)), dtype=torch.float64, device=target.device) if want_chi2 else None
    _check(lib().sm_solve_weights(arr, C.c_int(len(blocks)), C.c_int32(n_orb), _ptr(target), _ptr(sigma), _ptr(xi),
                                  C.c_int32(n_rhs), _ptr(keep), _ptr(wtilde), C.c_double(lam), C.c_double(rho),
                                  C.c_int32(n_iter), _ptr(w), _ptr(resid), _ptr(chi2), _stream(stream)), "sm_solve_weights")
    return {"w": w, "resid": resid, "chi2": chi2}


def sm_marginal_chi2(chi2, block_mask, stream=None):
    """Eq. 5-6: chi2 [n_rhs][n_blocks] CUDA f64 from sm_solve_weights -> tensor [2] = (chi2_model, chi2_min)."""
    import torch
    out = torch.empty(2, dtype=torch.float64, device=chi2.device)
    _check(lib().sm_marginal_chi2(_ptr(chi2), C.c_int32(chi2.shape[0]), C.c_int(chi2.shape[1]), C.c_uint32(block_mask), _ptr(out),
                                  _stream(stream)), "sm_marginal_chi2")
    return out


def sm_debug_gemm_f64(A, B, b_kmajor, alpha=1.0, beta=0.0, C_in=None, split_k=1, stream=None):
    """C = alpha * A @ (B.T if b_kmajor else B) + beta * C_in on CUDA float64 2-D tensors (row pitches from strides)."""
    import torch
    M, K = A.shape
    N = B.shape[0] if b_kmajor else B.shape[1]
    if split_k > 1:
        out = torch.empty((split_k, M, N), dtype=torch.float64, device=A.device)
        ldc = N
    else:
        out = C_in if C_in is not None else torch.empty((M, N), dtype=torch.float64, device=A.device)
        ldc = out.stride(0)
    _check(lib().sm_debug_gemm_f64(C.c_int(int(b_kmajor)), C.c_int(M), C.c_int(N), C.c_int(K), C.c_double(alpha), _ptr(A),
                                   C.c_int64(A.stride(0)), _ptr(B), C.c_int64(B.stride(0)), C.c_double(beta), _ptr(out),
                                   C.c_int64(ldc), C.c_int(split_k), _stream(stream)), "sm_debug_gemm_f64")
    return out


def sm_debug_invert_spd(A, stream=None):
    """In-place inverse of a CUDA float64 SPD matrix (rows may be padded: pitch = stride(0))."""
    _check(lib().sm_debug_invert_spd(_ptr(A), C.c_int64(A.stride(0)), C.c_int(A.shape[0]), _stream(stream)), "sm_debug_invert_spd")
    return A


def sm_set_debug_flags(flags):
    return lib().sm_set_debug_flags(C.c_int(flags))


def sm_measure_fma_peak(precision="f64", iters=20000):
    out = C.c_double()
    _check(lib().sm_measure_fma_peak(C.c_int(PRECISION[precision]), C.c_int(iters), C.byref(out)), "sm_measure_fma_peak")
    return out.value


def sm_last_kernel_times():
    """-> dict(phase_ms, integrate_ms, rowbuild_ms, zero_fill_ms) of the last build call made with debug flag 4."""
    out = (C.c_double * 4)()
    _check(lib().sm_last_kernel_times(out), "sm_last_kernel_times")
    return {"phase_ms": out[0], "integrate_ms": out[1], "rowbuild_ms": out[2], "zero_fill_ms": out[3]}


def sm_last_solve_times():
    """-> dict(setup_ms, inverse_ms, iterate_ms, xupdate_sampled_ms) of the last sm_solve_weights call made with debug flag 4."""
    out = (C.c_double * 4)()
    _check(lib().sm_last_solve_times(out), "sm_last_solve_times")
    return {"setup_ms": out[0], "inverse_ms": out[1], "iterate_ms": out[2], "xupdate_sampled_ms": out[3]}


def sm_launch_count():
    return int(lib().sm_launch_count())


def sm_version():
    return lib().sm_version()


def sm_debug_host_force(spec, xyz, t=0.0, precision="f64"):
    """Host-compiled copy of the kernels' force code, for CPU-side tests of tables and algebra only."""
    xyz = np.ascontiguousarray(xyz, dtype=np.float64).reshape(-1, 3)
    F, Phi = np.empty_like(xyz), np.empty(len(xyz))
    d = _desc(spec)
    _check(lib().sm_debug_host_force(C.byref(d), xyz.ctypes.data_as(C.c_void_p), C.c_int64(len(xyz)), C.c_double(t),
                                     C.c_int(PRECISION[precision]), F.ctypes.data_as(C.c_void_p),
                                     Phi.ctypes.data_as(C.c_void_p)), "sm_debug_host_force")
    return F, Phi


def sm_debug_host_lambda(a, b, c, xyz, guess):
    """Host-compiled copy of the kernels' Ferrers lambda iteration (fp32) with a warm-start guess per point (< 0: cold)."""
    xyz = np.ascontiguousarray(xyz, dtype=np.float64).reshape(-1, 3)
    guess = np.ascontiguousarray(guess, dtype=np.float32)
    lam, iters = np.empty(len(xyz), np.float32), np.empty(len(xyz), np.int32)
    _check(lib().sm_debug_host_lambda(C.c_double(a), C.c_double(b), C.c_double(c), xyz.ctypes.data_as(C.c_void_p),
                                      C.c_int64(len(xyz)), guess.ctypes.data_as(C.c_void_p), lam.ctypes.data_as(C.c_void_p),
                                      iters.ctypes.data_as(C.c_void_p)), "sm_debug_host_lambda")
    return lam, iters
