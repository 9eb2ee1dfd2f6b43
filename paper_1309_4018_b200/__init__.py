"""paper_1309_4018_b200 -- B200-native treecode BEM matvec / GMRES for the Poisson-Boltzmann equation.

Thin Python binding of the C ABI in include/pygbe.h (same names, argument marshalling only).  All
arithmetic runs in the CUDA kernels of libpygbe.so; PyTorch is used for device memory and streams.
There is no CPU fallback: importing works without a GPU (so that the build and the symbol table can
be checked), but any compute call without the library or a device raises.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpygbe.so")
HEADER_PATH = os.path.join(_HERE, "..", "include", "pygbe.h")

PYGBE_OK, PYGBE_EINVAL, PYGBE_ENOMEM, PYGBE_ECUDA, PYGBE_ENOCONV = 0, -1, -2, -3, -4
PRECISION_FP64, PRECISION_MIXED = 0, 1


class PygbeError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"pygbe error {code}: {msg}")
        self.code = code


class pygbe_surface(C.Structure):
    _fields_ = [("vertices", C.POINTER(C.c_double)), ("n_vertices", C.c_int64),
                ("triangles", C.POINTER(C.c_int32)), ("n_triangles", C.c_int64),
                ("region_in", C.c_int32), ("region_out", C.c_int32)]


class pygbe_charges(C.Structure):
    _fields_ = [("xyz", C.POINTER(C.c_double)), ("q", C.POINTER(C.c_double)),
                ("region", C.POINTER(C.c_int32)), ("n", C.c_int64)]


class pygbe_options(C.Structure):
    _fields_ = [("K_fine", C.c_int32), ("thres", C.c_double), ("N_k", C.c_int32), ("ncrit", C.c_int32),
                ("precision", C.c_int32), ("device", C.c_int32), ("stream", C.c_void_p),
                ("check_mesh", C.c_int32), ("precond", C.c_int32), ("group_mac", C.c_int32),
                ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t), ("reserved", C.c_int32 * 4)]


class pygbe_stats_t(C.Structure):
    _fields_ = [(n, C.c_int64) for n in (
        "n_panels", "n_unknowns", "n_regions", "n_surfaces", "n_charges", "n_points", "n_cells", "n_leaves",
        "n_groups", "tree_depth", "p2p_pairs", "m2p_evals", "direct_equiv", "near_nnz", "device_bytes",
        "workspace_high_water", "n_matvec", "kernels_per_matvec", "kernel_launches", "graph_launches")] + [
        ("create_ms", C.c_double), ("last_solve_ms", C.c_double), ("last_iters", C.c_int32),
        ("P", C.c_int32), ("K", C.c_int32), ("precision", C.c_int32), ("theta", C.c_double)]


class pygbe_launch_info(C.Structure):
    _fields_ = [("stage", C.c_int32), ("region", C.c_int32), ("twin_region", C.c_int32), ("launches", C.c_int32),
                ("ms", C.c_double), ("units", C.c_int64), ("bytes", C.c_int64), ("kernel", C.c_char * 64)]


_lib = None


def lib():
    """Load libpygbe.so (built in-tree by paper_1309_4018_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not found: run `python -m paper_1309_4018_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, dp, ip = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int32)
    L.pygbe_create.argtypes = [C.POINTER(pygbe_surface), C.c_int32, C.POINTER(pygbe_charges), dp, dp, C.c_int32,
                               C.c_int32, C.c_int32, C.c_double, C.POINTER(pygbe_options), C.POINTER(vp)]
    L.pygbe_workspace_size.argtypes = L.pygbe_create.argtypes[:-1] + [C.c_int32, C.POINTER(C.c_size_t)]
    L.pygbe_launch_times.argtypes = [vp, C.POINTER(pygbe_launch_info), C.c_int32, ip]
    L.pygbe_destroy.argtypes = [vp]
    L.pygbe_destroy.restype = None
    L.pygbe_num_unknowns.argtypes = [vp]
    L.pygbe_num_unknowns.restype = C.c_int64
    L.pygbe_matvec.argtypes = [vp, vp, vp]
    L.pygbe_matvec_host.argtypes = [vp, dp, dp]
    L.pygbe_rhs.argtypes = [vp, vp]
    L.pygbe_solve.argtypes = [vp, C.c_double, C.c_int32, C.c_int32, vp, ip, dp]
    L.pygbe_solve_host.argtypes = [vp, C.c_double, C.c_int32, C.c_int32, dp, ip, dp, dp, dp]
    L.pygbe_energy.argtypes = [vp, vp, dp, dp]
    L.pygbe_reaction_potential.argtypes = [vp, vp, vp]
    L.pygbe_stats.argtypes = [vp, C.POINTER(pygbe_stats_t)]
    L.pygbe_profile.argtypes = [vp, C.c_int]
    L.pygbe_stage_times.argtypes = [vp, dp, C.POINTER(C.c_int64)]
    L.pygbe_last_error.restype = C.c_char_p
    L.pygbe_version.restype = C.c_char_p
    _lib = L
    return L


def _check(rc, allow=()):
    if rc != PYGBE_OK and rc not in allow:
        raise PygbeError(rc, lib().pygbe_last_error().decode())
    return rc


def _dptr(t):
    """Device pointer of a contiguous fp64 CUDA torch tensor."""
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise TypeError("expected a contiguous float64 CUDA tensor")
    return C.c_void_p(t.data_ptr())


class Handle:
    """Owner of a pygbe_handle.  Methods mirror the C entry points one to one."""

    def __init__(self, surfaces, charges, eps, kappa, K=4, P=6, theta=0.5, K_fine=0, thres=0.0, N_k=0, ncrit=0,
                 precision=PRECISION_FP64, device=0, stream=None, check_mesh=False, precond=0, group_mac=0,
                 workspace="torch", gmres_restart=100):
        """surfaces: list of (vertices [nv,3] f64, triangles [nt,3] i32, region_in, region_out);
        charges: (xyz [nq,3], q [nq], region [nq] or None) or None.
        workspace: "torch" (default) -- query pygbe_workspace_size, allocate that block as a torch uint8 tensor
        and hand it to pygbe_create, so that every byte of the handle lives in torch's allocator; a uint8 CUDA
        tensor -- use it as the block; None -- let the library use its own pool.  gmres_restart sizes the GMRES
        buffers inside the block."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("pygbe needs a CUDA device (there is no CPU fallback)")
        L = lib()
        self._keep = []
        arr = (pygbe_surface * len(surfaces))()
        for i, (v, t, rin, rout) in enumerate(surfaces):
            v = np.ascontiguousarray(v, dtype=np.float64)
            t = np.ascontiguousarray(t, dtype=np.int32)
            self._keep += [v, t]
            arr[i] = pygbe_surface(v.ctypes.data_as(C.POINTER(C.c_double)), v.shape[0],
                                   t.ctypes.data_as(C.POINTER(C.c_int32)), t.shape[0], int(rin), int(rout))
        ch = None
        if charges is not None and len(charges[1]) > 0:
            xyz = np.ascontiguousarray(charges[0], dtype=np.float64).reshape(-1, 3)
            q = np.ascontiguousarray(charges[1], dtype=np.float64).reshape(-1)
            reg = None
            if len(charges) > 2 and charges[2] is not None:
                reg = np.ascontiguousarray(charges[2], dtype=np.int32).reshape(-1)
            self._keep += [xyz, q, reg]
            ch = pygbe_charges(xyz.ctypes.data_as(C.POINTER(C.c_double)), q.ctypes.data_as(C.POINTER(C.c_double)),
                               reg.ctypes.data_as(C.POINTER(C.c_int32)) if reg is not None else None, q.shape[0])
        eps = np.ascontiguousarray(eps, dtype=np.float64)
        kappa = np.ascontiguousarray(kappa, dtype=np.float64)
        if stream is None:
            stream = torch.cuda.current_stream(device).cuda_stream
        opt = pygbe_options(K_fine=K_fine, thres=thres, N_k=N_k, ncrit=ncrit, precision=precision, device=device,
                            stream=C.c_void_p(stream), check_mesh=int(check_mesh), precond=int(precond),
                            group_mac=int(group_mac))
        args = (arr, len(surfaces), C.byref(ch) if ch is not None else None,
                eps.ctypes.data_as(C.POINTER(C.c_double)), kappa.ctypes.data_as(C.POINTER(C.c_double)),
                len(eps), K, P, float(theta), C.byref(opt))
        self.workspace = None
        self.workspace_query_ms = 0.0
        if isinstance(workspace, str):
            if workspace != "torch":
                raise ValueError("workspace must be 'torch', a uint8 CUDA tensor or None")
            import time
            t0 = time.perf_counter()
            nbytes = C.c_size_t()
            _check(L.pygbe_workspace_size(*args, int(gmres_restart), C.byref(nbytes)))
            self.workspace_query_ms = 1e3 * (time.perf_counter() - t0)
            workspace = torch.empty(nbytes.value, dtype=torch.uint8, device=torch.device("cuda", device))
        if workspace is not None:
            if not (isinstance(workspace, torch.Tensor) and workspace.is_cuda and workspace.dtype == torch.uint8
                    and workspace.is_contiguous()):
                raise TypeError("workspace must be a contiguous uint8 CUDA tensor")
            self.workspace = workspace                     # keeps the block alive as long as the handle
            opt.workspace = C.c_void_p(workspace.data_ptr())
            opt.workspace_bytes = workspace.numel()
        h = C.c_void_p()
        _check(L.pygbe_create(*args, C.byref(h)))
        self._h = h
        self.device = torch.device("cuda", device)
        self.n = int(L.pygbe_num_unknowns(h))
        self._keep = []

    @classmethod
    def from_problem(cls, p, **kw):
        """Build from a workloads.Problem-like object (surfaces, eps, kappa, charge_* attributes)."""
        surfaces = [(s.vertices, s.triangles, s.region_in, s.region_out) for s in p.surfaces]
        return cls(surfaces, (p.charge_xyz, p.charge_q, p.charge_region), p.eps, p.kappa, **kw)

    @staticmethod
    def workspace_size(p, gmres_restart=100, **kw):
        """pygbe_workspace_size for a workloads.Problem-like object and the keyword arguments of Handle."""
        kw = dict(kw, workspace=None)
        return _workspace_size_of(p, gmres_restart, **kw)

    def close(self):
        if getattr(self, "_h", None):
            lib().pygbe_destroy(self._h)
            self._h = None
        self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def num_unknowns(self):
        return self.n

    def matvec(self, x, y=None):
        import torch
        if y is None:
            y = torch.empty(self.n, dtype=torch.float64, device=self.device)
        _check(lib().pygbe_matvec(self._h, _dptr(x), _dptr(y)))
        return y

    def matvec_host(self, x, y=None):
        x = np.ascontiguousarray(x, dtype=np.float64)
        if y is None:
            y = np.empty(self.n)
        dp = C.POINTER(C.c_double)
        _check(lib().pygbe_matvec_host(self._h, x.ctypes.data_as(dp), y.ctypes.data_as(dp)))
        return y

    def rhs(self, b=None):
        import torch
        if b is None:
            b = torch.empty(self.n, dtype=torch.float64, device=self.device)
        _check(lib().pygbe_rhs(self._h, _dptr(b)))
        return b

    def solve(self, tol=1e-6, restart=100, max_iter=1000, x=None, raise_on_noconv=True):
        import torch
        if x is None:
            x = torch.empty(self.n, dtype=torch.float64, device=self.device)
        it = C.c_int32(); rel = C.c_double()
        rc = _check(lib().pygbe_solve(self._h, tol, restart, max_iter, _dptr(x), C.byref(it), C.byref(rel)),
                    allow=() if raise_on_noconv else (PYGBE_ENOCONV,))
        return x, it.value, rel.value, rc

    def solve_host(self, tol=1e-6, restart=100, max_iter=1000, want_x=True):
        x = np.empty(self.n) if want_x else None
        it = C.c_int32(); rel = C.c_double(); es = C.c_double(); ec = C.c_double()
        dp = C.POINTER(C.c_double)
        _check(lib().pygbe_solve_host(self._h, tol, restart, max_iter, x.ctypes.data_as(dp) if want_x else None,
                                      C.byref(it), C.byref(rel), C.byref(es), C.byref(ec)))
        return x, it.value, rel.value, es.value, ec.value

    def energy(self, x):
        es = C.c_double(); ec = C.c_double()
        _check(lib().pygbe_energy(self._h, _dptr(x), C.byref(es), C.byref(ec)))
        return es.value, ec.value

    def reaction_potential(self, x, n_charges):
        import torch
        phi = torch.empty(n_charges, dtype=torch.float64, device=self.device)
        _check(lib().pygbe_reaction_potential(self._h, _dptr(x), _dptr(phi)))
        return phi

    STAGES = ("prep", "p2m", "m2m", "m2p", "p2p", "near", "combine", "reserved")

    def profile(self, enable=True):
        _check(lib().pygbe_profile(self._h, int(bool(enable))))

    def stage_times(self):
        """{stage: (accumulated ms, kernel launches)} since profile(True)."""
        ms = (C.c_double * 8)()
        ln = (C.c_int64 * 8)()
        _check(lib().pygbe_stage_times(self._h, ms, ln))
        return {name: (ms[i], ln[i]) for i, name in enumerate(self.STAGES) if name != "reserved"}

    def launch_times(self):
        """Per kernel launch of the matvec since profile(True): list of dicts (stage, region, twin_region,
        launches, ms, units, bytes, kernel); ms is accumulated over `launches` launches."""
        buf = (pygbe_launch_info * 64)()
        n = C.c_int32()
        _check(lib().pygbe_launch_times(self._h, buf, 64, C.byref(n)))
        return [dict(stage=self.STAGES[b.stage], region=b.region, twin_region=b.twin_region, launches=b.launches, ms=b.ms,
                     units=b.units, bytes=b.bytes, kernel=b.kernel.decode()) for b in buf[:n.value]]

    def stats(self):
        s = pygbe_stats_t()
        _check(lib().pygbe_stats(self._h, C.byref(s)))
        return {name: getattr(s, name) for name, _ in pygbe_stats_t._fields_}


def _workspace_size_of(p, gmres_restart, **kw):
    """Marshalling for Handle.workspace_size (the arrays only need to live for the duration of the call)."""
    L = lib()
    surfaces = [(s.vertices, s.triangles, s.region_in, s.region_out) for s in p.surfaces]
    keep = []
    arr = (pygbe_surface * len(surfaces))()
    for i, (v, t, rin, rout) in enumerate(surfaces):
        v = np.ascontiguousarray(v, dtype=np.float64); t = np.ascontiguousarray(t, dtype=np.int32)
        keep += [v, t]
        arr[i] = pygbe_surface(v.ctypes.data_as(C.POINTER(C.c_double)), v.shape[0],
                               t.ctypes.data_as(C.POINTER(C.c_int32)), t.shape[0], int(rin), int(rout))
    ch = None
    if len(p.charge_q) > 0:
        xyz = np.ascontiguousarray(p.charge_xyz, dtype=np.float64).reshape(-1, 3)
        q = np.ascontiguousarray(p.charge_q, dtype=np.float64).reshape(-1)
        reg = np.ascontiguousarray(p.charge_region, dtype=np.int32).reshape(-1)
        keep += [xyz, q, reg]
        ch = pygbe_charges(xyz.ctypes.data_as(C.POINTER(C.c_double)), q.ctypes.data_as(C.POINTER(C.c_double)),
                           reg.ctypes.data_as(C.POINTER(C.c_int32)), q.shape[0])
    eps = np.ascontiguousarray(p.eps, dtype=np.float64); kappa = np.ascontiguousarray(p.kappa, dtype=np.float64)
    K, P, theta = kw.pop("K", 4), kw.pop("P", 6), kw.pop("theta", 0.5)
    kw.pop("workspace", None); kw.pop("stream", None)
    opt = pygbe_options(**{k: (int(v) if k != "thres" else float(v)) for k, v in kw.items()})
    nbytes = C.c_size_t()
    _check(L.pygbe_workspace_size(arr, len(surfaces), C.byref(ch) if ch is not None else None,
                                  eps.ctypes.data_as(C.POINTER(C.c_double)), kappa.ctypes.data_as(C.POINTER(C.c_double)),
                                  len(eps), K, P, float(theta), C.byref(opt), int(gmres_restart), C.byref(nbytes)))
    return nbytes.value


def alu_peaks(device=0):
    """Measured ALU peaks of the device: dict(fp32_tflops, fp64_tflops, mufu_gops, fp32_mix_tflops, fp32_horner_tflops)."""
    L = lib()
    L.pygbe_alu_peaks.argtypes = [C.c_int32, C.POINTER(C.c_double)]
    out = (C.c_double * 5)()
    _check(L.pygbe_alu_peaks(device, out))
    return dict(fp32_tflops=out[0], fp64_tflops=out[1], mufu_gops=out[2], fp32_mix_tflops=out[3], fp32_horner_tflops=out[4])


def mma_probe(P=8, device=0):
    """pygbe_mma_probe: {variant: dict(ms, rel_l2, pairs)} for the CUDA-core M2P, the monomial-tile write alone and the
    TF32 tensor-core contraction in one pass and with the 3 x TF32 split (csrc/mma_probe.cuh)."""
    L = lib()
    L.pygbe_mma_probe.argtypes = [C.c_int32, C.c_int32, C.POINTER(C.c_double)]
    out = (C.c_double * 12)()
    _check(L.pygbe_mma_probe(device, P, out))
    names = ("cuda_core_k_m2p_single2", "monomial_tile_to_smem_only", "tile_plus_tf32_mma_1pass", "tile_plus_tf32_mma_3xsplit")
    return {n: dict(ms=out[3 * i], rel_l2=out[3 * i + 1], pairs=out[3 * i + 2]) for i, n in enumerate(names)}


NOALLOC_MAX_CHARGES = 16384


def coulomb_energy_noalloc(xyz, q, eps, out, device=0, stream=None):
    """pygbe_coulomb_energy_noalloc: Coulomb energy (kJ/mol) of the charges xyz [n,3], q [n] (fp64 CUDA tensors) in a
    region of permittivity eps, written to out (fp64 CUDA tensor, 1 element).  Allocates nothing; asynchronous."""
    import torch
    L = lib()
    L.pygbe_coulomb_energy_noalloc.argtypes = [C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_double, C.c_void_p]
    if stream is None:
        stream = torch.cuda.current_stream(device).cuda_stream
    n = int(q.numel())
    _check(L.pygbe_coulomb_energy_noalloc(device, C.c_void_p(stream), _dptr(xyz) if n else None, _dptr(q) if n else None, n,
                                          float(eps), _dptr(out)))
    return out


def noalloc_setup(device=0):
    L = lib()
    L.pygbe_noalloc_setup.argtypes = [C.c_int32]
    _check(L.pygbe_noalloc_setup(device))


def host_table(which, P, kappa=0.0):
    """pygbe_host_table: (off, k, c, deg) of the M2P coefficient table (0: regrouped / reduced, 1: Laplace form).  No GPU."""
    L = lib()
    ip = C.POINTER(C.c_int32)
    L.pygbe_host_table.argtypes = [C.c_int32, C.c_int32, C.c_double, C.c_int32, C.c_int32, ip, ip, ip, C.POINTER(C.c_int16),
                                   C.POINTER(C.c_double), C.POINTER(C.c_int16)]
    ne, nz = C.c_int32(), C.c_int32()
    _check(L.pygbe_host_table(which, P, float(kappa), 0, 0, C.byref(ne), C.byref(nz), None, None, None, None))
    off = np.zeros(ne.value + 1, dtype=np.int32); k = np.zeros(nz.value, dtype=np.int16)
    c = np.zeros(nz.value); deg = np.zeros(ne.value, dtype=np.int16)
    _check(L.pygbe_host_table(which, P, float(kappa), ne.value, nz.value, C.byref(ne), C.byref(nz), off.ctypes.data_as(ip),
                              k.ctypes.data_as(C.POINTER(C.c_int16)), c.ctypes.data_as(C.POINTER(C.c_double)),
                              deg.ctypes.data_as(C.POINTER(C.c_int16))))
    return off, k, c, deg


def pygbe_version():
    return lib().pygbe_version().decode()
