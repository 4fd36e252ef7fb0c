"""f4: slab-decomposed complex 3D transform over several GPUs.

One process per GPU.  Rank r holds the z slab [Nz/R][Ny][Nx] of a field in real space and the y slab [Nz][Ny/R][Nx] of
its transform.  The transpose between the two is the store phase of the pass that precedes it: the kernels write
straight into the peers' slabs, which every rank has mapped through CUDA IPC (NVLink peer memory) -- `torch.distributed`
carries only the 64-byte handles at set-up and one barrier per transform.  Argument marshalling and plumbing only: the
passes run in the library's kernels (include/arche.h: arche_fft3d_slab_scatter / arche_fft3d_slab_finish).

`slab_ranges`, `exchange_handles` and `SlabPlan` hold the host logic and need no GPU (gloo tests); `SlabFFT` is the
device object; `VirtualSlabs` runs R slabs on ONE GPU one after the other (each kernel completes before the next
starts; nothing waits on a peer) -- the single-GPU parity test of the decomposition."""
from __future__ import annotations

import ctypes as C


def slab_ranges(n: int, world: int):
    """[lo, hi) of every rank along an axis of length n; n must be a multiple of world (the kernels' requirement)"""
    if world < 1 or n % world:
        raise ValueError(f"axis length {n} is not a multiple of {world} ranks")
    w = n // world
    return [(r * w, (r + 1) * w) for r in range(world)]


class SlabPlan:
    """sizes and index maps of the decomposition (pure host arithmetic)"""

    def __init__(self, grid, world: int, rank: int):
        self.nx, self.ny, self.nz = (int(g) for g in grid)
        self.world, self.rank = int(world), int(rank)
        if not 0 <= self.rank < self.world or self.world > 16:
            raise ValueError("rank outside the world, or more than 16 ranks")
        self.z_lo, self.z_hi = slab_ranges(self.nz, world)[rank]
        self.y_lo, self.y_hi = slab_ranges(self.ny, world)[rank]
        self.nzl, self.nyl = self.z_hi - self.z_lo, self.y_hi - self.y_lo
        self.z_slab_shape = (self.nzl, self.ny, self.nx)
        self.y_slab_shape = (self.nz, self.nyl, self.nx)
        self.slab_elems = self.nzl * self.ny * self.nx        # = nz * nyl * nx
        self.slab_bytes = 16 * self.slab_elems

    def owner_after_forward(self, iy: int) -> int:
        return iy // self.nyl

    def owner_after_inverse(self, iz: int) -> int:
        return iz // self.nzl


def exchange_handles(handle: bytes, group=None):
    """all-gather of one opaque handle per rank, in rank order (torch.distributed, any backend)"""
    import torch.distributed as dist
    out = [None] * dist.get_world_size(group)
    dist.all_gather_object(out, bytes(handle), group=group)
    return out


class _Buffers:
    """two IPC-exportable slab buffers (z slab, y slab) + scratch on the current device"""

    def __init__(self, lib, nbytes):
        self.lib, self.ptrs = lib, []
        for _ in range(3):
            p = C.c_void_p()
            if lib.arche_slab_alloc(nbytes, C.byref(p)) != 0:
                raise MemoryError("arche_slab_alloc failed")
            self.ptrs.append(p.value)
        self.z, self.y, self.scratch = self.ptrs

    def free(self):
        for p in self.ptrs:
            self.lib.arche_slab_free(p)
        self.ptrs = []


class SlabFFT:
    """One rank of the decomposed transform.  `ctx` is an `Arche` context of the GLOBAL grid on this rank's GPU."""

    def __init__(self, ctx, group=None):
        import torch
        import torch.distributed as dist
        self.torch, self.ctx, self.group = torch, ctx, group
        self.world, self.rank = dist.get_world_size(group), dist.get_rank(group)
        self.plan = SlabPlan(ctx.grid, self.world, self.rank)
        self.buf = _Buffers(ctx.lib, self.plan.slab_bytes)
        hz, hy = C.create_string_buffer(64), C.create_string_buffer(64)
        ctx._check(ctx.lib.arche_ipc_export(self.buf.z, hz)); ctx._check(ctx.lib.arche_ipc_export(self.buf.y, hy))
        self.peer_z, self.peer_y, self._opened = [], [], []
        for which, mine, handles in (("z", self.buf.z, exchange_handles(hz.raw, group)), ("y", self.buf.y, exchange_handles(hy.raw, group))):
            for q, h in enumerate(handles):
                if q == self.rank:
                    ptr = mine
                else:
                    p = C.c_void_p()
                    ctx._check(ctx.lib.arche_ipc_open(h, C.byref(p)))
                    ptr = p.value; self._opened.append(ptr)
                (self.peer_z if which == "z" else self.peer_y).append(ptr)

    def _view(self, ptr, shape):
        n = shape[0] * shape[1] * shape[2]

        class _A:   # a tensor over library-owned memory (no copy) through the __cuda_array_interface__ protocol
            __cuda_array_interface__ = {"shape": (n,), "typestr": "<c16", "data": (int(ptr), False), "version": 3}
        return self.torch.as_tensor(_A(), device=self.ctx.device).view(shape)

    def z_slab(self):
        return self._view(self.buf.z, self.plan.z_slab_shape)

    def y_slab(self):
        return self._view(self.buf.y, self.plan.y_slab_shape)

    def _barrier(self):
        import torch.distributed as dist
        self.ctx.sync()
        dist.barrier(group=self.group)

    def forward(self):
        """z slab (buffer z_slab()) -> y slab of the transform (buffer y_slab()), sign -1, unnormalised"""
        self._barrier()                        # nobody still reads the y slabs of a previous transform
        self.ctx.fft3d_slab_scatter(self.buf.z, self.buf.scratch, self.peer_y, self.rank, -1)
        self._barrier()                        # every rank's rows have landed
        self.ctx.fft3d_slab_finish(self.buf.y, self.world, -1)
        self.ctx.sync()

    def inverse(self):
        """y slab -> z slab, sign +1, unnormalised"""
        self._barrier()
        self.ctx.fft3d_slab_scatter(self.buf.y, None, self.peer_z, self.rank, +1)
        self._barrier()
        self.ctx.fft3d_slab_finish(self.buf.z, self.world, +1)
        self.ctx.sync()

    def close(self):
        for p in self._opened:
            self.ctx.lib.arche_ipc_close(p)
        self._opened = []
        self.buf.free()


class VirtualSlabs:
    """R slabs on ONE GPU, processed one after the other through the same two entry points: every kernel has completed
    before the next "rank" starts, so nothing ever waits on a peer.  Checks the decomposition (index maps of the scatter
    stores, slab-local passes) against the undecomposed transform; says nothing about NVLink."""

    def __init__(self, ctx, world: int):
        import torch
        self.torch, self.ctx, self.world = torch, ctx, int(world)
        self.plans = [SlabPlan(ctx.grid, world, r) for r in range(world)]
        p0 = self.plans[0]
        dev = ctx.device
        self.z = [torch.zeros(p0.z_slab_shape, dtype=torch.complex128, device=dev) for _ in range(world)]
        self.y = [torch.zeros(p0.y_slab_shape, dtype=torch.complex128, device=dev) for _ in range(world)]
        self.scratch = torch.empty(p0.z_slab_shape, dtype=torch.complex128, device=dev)

    def load(self, field):
        """field: [nz][ny][nx] complex (host or device) -> z slabs"""
        f = self.torch.as_tensor(field, device=self.ctx.device).to(self.torch.complex128)
        for r, p in enumerate(self.plans):
            self.z[r].copy_(f[p.z_lo:p.z_hi])

    def forward(self):
        for r in range(self.world):
            self.ctx.fft3d_slab_scatter(self.z[r].data_ptr(), self.scratch.data_ptr(), [t.data_ptr() for t in self.y], r, -1)
            self.ctx.sync()
        for r in range(self.world):
            self.ctx.fft3d_slab_finish(self.y[r].data_ptr(), self.world, -1)
        self.ctx.sync()

    def inverse(self):
        for r in range(self.world):
            self.ctx.fft3d_slab_scatter(self.y[r].data_ptr(), None, [t.data_ptr() for t in self.z], r, +1)
            self.ctx.sync()
        for r in range(self.world):
            self.ctx.fft3d_slab_finish(self.z[r].data_ptr(), self.world, +1)
        self.ctx.sync()

    def spectrum(self):
        """the y slabs gathered into the full [nz][ny][nx] spectrum"""
        return self.torch.cat(self.y, dim=1)

    def field(self):
        return self.torch.cat(self.z, dim=0)
