"""One periodic N^3 lattice sharded into z slabs over several GPUs (include/prs.h, "z slabs").

SURVEY.md 8(e) / 8(f4); PAPER.md:141-143 names device memory as the limit on the box size.  Every
step of the path still runs in the kernels of libprs: a slab handle advances its owned planes plus four
halo planes per side, and what this module adds is only the transport of the halo planes between
slabs (contiguous blocks of 4*N*N values of phi and of phidot, one per direction and field, once per
four steps) and the sum of the slabs' diagnostics:

``SlabSimulation``      the C calls of one slab (``prs_create_slab`` ... ``prs_slab_halo_filled``).
``exchange_halo_tensors``  the halo transport over ``torch.distributed`` point-to-point operations
                        (NCCL over NVLink between GPUs; gloo in the CPU tests of the plumbing).
``ShardedSimulation``   one rank of a ``torch.distributed`` job: slab ``rank`` of ``world`` equal slabs.
``SlabGroup``           all slabs driven by ONE process, each on a device of its own (or several on one
                        device): halo planes move by peer-to-peer ``copy_`` ordered by CUDA events.

The owned planes of the slabs are bit-identical to the unsharded lattice at every step (each site sees
the same operations); link and wall-site counts add up exactly; the velocity sum differs from the
unsharded one only by the order of its double additions.
"""
import ctypes as C

from .prs import F32, INFO_KERNEL_LAUNCHES, PrsError, Simulation, diag_combine, lib

INFO_HALO_VALID, INFO_HALO_PLANES = 5, 6
HALO = 4                       # planes per side; also the steps of one pass of the four-step kernel


def _slab_lib():
    L = lib()
    if not getattr(L, "_slab_ready", False):
        vp, i64, dbl, u64, ci, sz = C.c_void_p, C.c_int64, C.c_double, C.c_uint64, C.c_int, C.c_size_t
        L.prs_slab_workspace_bytes.argtypes = [i64, i64, ci]
        L.prs_slab_workspace_bytes.restype = sz
        L.prs_create_slab.argtypes = [C.POINTER(vp), i64, i64, i64, ci, dbl, dbl, dbl, dbl, dbl, u64, vp, sz, vp]
        L.prs_slab_halo_regions.argtypes = [vp, vp * 4, vp * 4, C.POINTER(sz)]
        L.prs_slab_halo_filled.argtypes = [vp]
        L._slab_ready = True
    return L


def slab_bounds(N, world, rank):
    """(z_begin, nz) of slab ``rank`` of ``world`` equal slabs; N must divide evenly into slabs of >= 4 planes."""
    if world < 1 or not 0 <= rank < world:
        raise ValueError("need 0 <= rank < world")
    if N % world != 0 or N // world < HALO:
        raise ValueError("N = %d does not split into %d equal slabs of at least %d planes" % (N, world, HALO))
    nz = N // world
    return rank * nz, nz


def step_schedule(nsteps, halo_valid):
    """The launches of ``nsteps`` steps on a slab whose halo is good for ``halo_valid`` more steps:
    a list of ("exchange",) and ("step", k) with k <= 4.  Whole passes of four steps first (each after
    an exchange unless the halo is still fresh), then the remainder."""
    out, left, valid = [], int(nsteps), int(halo_valid)
    while left > 0:
        k = min(left, HALO)
        if valid < k:
            out.append(("exchange",))
            valid = HALO
        out.append(("step", k))
        valid -= k
        left -= k
    return out


class SlabSimulation(Simulation):
    """One z slab [z_begin, z_begin + nz) of a periodic N^3 lattice on one device (prs_create_slab)."""

    def __init__(self, N, z_begin, nz, precision=F32, alpha=3.0, era_m=1.0, deta=0.1, W0=10.0, phi0=1.0, seed=1,
                 device=None, stream=None):
        import torch  # device memory and streams only

        if not torch.cuda.is_available():
            raise RuntimeError("paper_1710_10420_b200 needs a CUDA device (no CPU fallback)")
        L = _slab_lib()
        self._torch = torch
        self.dims, self.N, self.precision = 3, int(N), int(precision)
        self.z_begin, self.nz = int(z_begin), int(nz)
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        self.dtype = torch.float32 if precision == F32 else torch.float64
        self.shape = (self.nz, self.N, self.N)
        nbytes = int(L.prs_slab_workspace_bytes(N, nz, precision))
        if nbytes == 0:
            raise PrsError(1, "prs_slab_workspace_bytes")
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self.stream = torch.cuda.current_stream(self.device) if stream is None else stream
            self._h = C.c_void_p()
            rc = L.prs_create_slab(C.byref(self._h), N, z_begin, nz, precision, alpha, era_m, deta, W0, phi0, seed,
                                   self.workspace.data_ptr(), nbytes, self.stream.cuda_stream)
        if rc != 0:
            self._h = C.c_void_p()
            raise PrsError(rc, "prs_create_slab")

    def copy_in(self, phi, phidot, eta0=1.0, step=0):
        import numpy as np

        dt = np.float32 if self.precision == F32 else np.float64
        a, b = np.ascontiguousarray(phi, dt), np.ascontiguousarray(phidot, dt)
        if a.size != self.nz * self.N * self.N or b.size != a.size:
            raise ValueError("arrays must hold the nz*N*N owned sites")
        self._chk(lib().prs_copy_in(self._h, a.ctypes.data, b.ctypes.data, eta0, step), "prs_copy_in")

    def halo_regions(self):
        """(send, recv): two lists of four uint8 views of the workspace -- phi low, phi high, phidot low,
        phidot high -- into the CURRENT arrays (ask again after every step)."""
        send, recv, nbytes = (C.c_void_p * 4)(), (C.c_void_p * 4)(), C.c_size_t()
        self._chk(_slab_lib().prs_slab_halo_regions(self._h, send, recv, C.byref(nbytes)), "prs_slab_halo_regions")
        base, n = self.workspace.data_ptr(), int(nbytes.value)
        view = lambda p: self.workspace[p - base:p - base + n]   # noqa: E731
        return [view(p) for p in send], [view(p) for p in recv]

    def halo_filled(self):
        self._chk(_slab_lib().prs_slab_halo_filled(self._h), "prs_slab_halo_filled")

    @property
    def halo_valid(self):
        return self.get_info(INFO_HALO_VALID)


def exchange_halo_tensors(send, recv, rank, world, group=None):
    """Moves the four halo blocks of one slab over ``torch.distributed``: send[2f] (field f's lowest owned
    planes) goes to rank-1's recv[2f+1] (its upper halo), send[2f+1] (highest owned planes) to rank+1's
    recv[2f] (its lower halo), periodically.  Every rank posts its operations in the same order -- per
    field: send down, send up, receive from above, receive from below -- so that with two ranks, where both
    neighbours are the same peer, the messages pair up by order (NCCL) as well as by tag (gloo)."""
    import torch.distributed as dist

    if world == 1:
        for f in range(len(send) // 2):
            recv[2 * f + 1].copy_(send[2 * f])
            recv[2 * f].copy_(send[2 * f + 1])
        return
    if send[0].is_cuda and dist.get_backend(group) == "gloo":
        # gloo moves host memory only: stage the blocks through the host (a transport for boxes without
        # NCCL between the ranks' GPUs, and for the two-ranks-on-one-GPU test)
        hs, hr = [t.cpu() for t in send], [t.new_empty(t.shape, device="cpu") for t in recv]
        exchange_halo_tensors(hs, hr, rank, world, group)
        for d, h in zip(recv, hr):
            d.copy_(h)
        return
    down, up = (rank - 1) % world, (rank + 1) % world
    if group is not None:
        down, up = dist.get_global_rank(group, down), dist.get_global_rank(group, up)
    ops = []
    for f in range(len(send) // 2):
        ops.append(dist.P2POp(dist.isend, send[2 * f], down, group=group, tag=2 * f))
        ops.append(dist.P2POp(dist.isend, send[2 * f + 1], up, group=group, tag=2 * f + 1))
        ops.append(dist.P2POp(dist.irecv, recv[2 * f + 1], up, group=group, tag=2 * f))
        ops.append(dist.P2POp(dist.irecv, recv[2 * f], down, group=group, tag=2 * f + 1))
    for req in dist.batch_isend_irecv(ops):
        req.wait()


def combine_diagnostics(parts, N):
    """The lattice's diagnostics from the slabs' partial sums (dicts of prs_diag fields): prs_diag_combine
    (the sums and the normalisation of Eqs. 7-8 are the library's, not this module's)."""
    return diag_combine(parts, 3, N)


class ShardedSimulation:
    """Slab ``rank`` of ``world`` equal z slabs, one process per GPU under ``torch.distributed``."""

    def __init__(self, N, precision=F32, group=None, rank=None, world=None, **kw):
        import torch
        import torch.distributed as dist

        self._torch, self._dist, self.group = torch, dist, group
        self.rank = dist.get_rank(group) if rank is None else rank
        self.world = dist.get_world_size(group) if world is None else world
        self.N = int(N)
        z_begin, nz = slab_bounds(self.N, self.world, self.rank)
        self.slab = SlabSimulation(N, z_begin, nz, precision, **kw)

    def init(self, eta0=1.0):
        self.slab.init(eta0)

    def exchange(self):
        """Halo transport on the slab's own stream: the blocks are read after the step kernels queued there and
        the next step is queued behind the copies, whatever torch's current stream is (torch.distributed's
        point-to-point operations and ``copy_`` order themselves against the CURRENT stream)."""
        torch = self._torch
        send, recv = self.slab.halo_regions()
        with torch.cuda.device(self.slab.device), torch.cuda.stream(self.slab.stream):
            exchange_halo_tensors(send, recv, self.rank, self.world, self.group)
        self.slab.halo_filled()

    def step(self, nsteps=1):
        for op in step_schedule(nsteps, self.slab.halo_valid):
            if op[0] == "exchange":
                self.exchange()
            else:
                self.slab.step(op[1])

    def diagnostics(self):
        """The whole lattice's diagnostics, on every rank."""
        torch, dist = self._torch, self._dist
        if self.slab.halo_valid < 1:
            self.exchange()
        d = self.slab.diagnostics()
        dev = self.slab.device if self.world > 1 and dist.get_backend(self.group) == "nccl" else "cpu"
        counts = torch.tensor([d["link_count"], d["wall_sites"]], dtype=torch.int64, device=dev)
        ratio = torch.tensor([d["sum_ratio"]], dtype=torch.float64, device=dev)
        if self.world > 1:
            dist.all_reduce(counts, group=self.group)
            dist.all_reduce(ratio, group=self.group)
        links, walls = (int(v) for v in counts.tolist())
        part = dict(d, link_count=links, wall_sites=walls, sum_ratio=float(ratio.item()))
        return combine_diagnostics([part], self.N)

    def weighted_area(self):
        """(area, rho_weighted) of the whole lattice (Eq. 7 with the orientation weight), on every rank."""
        torch, dist = self._torch, self._dist
        if self.slab.halo_valid < 1:
            self.exchange()
        area, _ = self.slab.weighted_area()
        if self.world > 1:
            dev = self.slab.device if dist.get_backend(self.group) == "nccl" else "cpu"
            t = torch.tensor([area], dtype=torch.float64, device=dev)
            dist.all_reduce(t, group=self.group)
            area = float(t.item())
        return area, area / float(self.N) ** 3

    def copy_out(self):
        """This rank's owned planes: two numpy arrays of shape (nz, N, N)."""
        return self.slab.copy_out()

    @property
    def kernel_launches(self):
        return self.slab.get_info(INFO_KERNEL_LAUNCHES)

    def close(self):
        self.slab.close()


class SlabGroup:
    """All slabs of one lattice driven by one process: slab r on ``devices[r]`` (devices may repeat --
    several slabs on one GPU run one after the other).  Halo planes move by ``copy_`` between the slabs'
    workspaces (peer-to-peer over NVLink between devices), ordered against the step kernels by CUDA events."""

    def __init__(self, N, devices, precision=F32, **kw):
        import torch

        self._torch, self.N, self.world = torch, int(N), len(devices)
        self.slabs = []
        for r, dev in enumerate(devices):
            z_begin, nz = slab_bounds(self.N, self.world, r)
            dev = torch.device("cuda", dev) if isinstance(dev, int) else torch.device(dev)
            with torch.cuda.device(dev):
                self.slabs.append(SlabSimulation(N, z_begin, nz, precision, device=dev, **kw))

    def init(self, eta0=1.0):
        for s in self.slabs:
            s.init(eta0)

    def exchange(self):
        torch = self._torch
        regions = [s.halo_regions() for s in self.slabs]
        done = [s.stream.record_event() for s in self.slabs]        # the steps that produced the planes
        copied = []
        for r, s in enumerate(self.slabs):
            down, up = (r - 1) % self.world, (r + 1) % self.world
            s.stream.wait_event(done[down])
            s.stream.wait_event(done[up])
            with torch.cuda.device(s.device), torch.cuda.stream(s.stream):
                for f in range(2):
                    regions[r][1][2 * f].copy_(regions[down][0][2 * f + 1], non_blocking=True)      # lower halo
                    regions[r][1][2 * f + 1].copy_(regions[up][0][2 * f], non_blocking=True)        # upper halo
            copied.append(s.stream.record_event())
        for r, s in enumerate(self.slabs):                             # nobody overwrites planes still being read
            s.stream.wait_event(copied[(r - 1) % self.world])
            s.stream.wait_event(copied[(r + 1) % self.world])
            s.halo_filled()

    def step(self, nsteps=1):
        for op in step_schedule(nsteps, min(s.halo_valid for s in self.slabs)):
            if op[0] == "exchange":
                self.exchange()
            else:
                for s in self.slabs:
                    s.step(op[1])

    def diagnostics(self):
        if min(s.halo_valid for s in self.slabs) < 1:
            self.exchange()
        return combine_diagnostics([s.diagnostics() for s in self.slabs], self.N)

    def weighted_area(self):
        """(area, rho_weighted) of the whole lattice: the slabs' partial sums added in slab order."""
        if min(s.halo_valid for s in self.slabs) < 1:
            self.exchange()
        area = 0.0
        for s in self.slabs:
            area += s.weighted_area()[0]
        return area, area / float(self.N) ** 3

    def copy_out(self):
        """The whole lattice: two numpy arrays of shape (N, N, N)."""
        import numpy as np

        parts = [s.copy_out() for s in self.slabs]
        return np.concatenate([p[0] for p in parts]), np.concatenate([p[1] for p in parts])

    @property
    def kernel_launches(self):
        return sum(s.get_info(INFO_KERNEL_LAUNCHES) for s in self.slabs)

    def close(self):
        for s in self.slabs:
            s.close()
