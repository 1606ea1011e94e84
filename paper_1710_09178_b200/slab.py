"""t-slab decomposition of the lattice over ranks: index maps, halo exchange and
the callbacks of the library's slab mode -- no operator or solver arithmetic lives here; the stencil is the
library's (qcd_dslash_range, or qcd_dslash / qcd_mdagm / qcd_multishift_cg after qcd_set_slab).

The paper slices the lattice along z, K computational slices plus halos per node, and exchanges the
faces before every D.  Here the slicing direction is t (the slowest
index of the canonical address l = ((t*Nz + z)*Ny + y)*Nx + x, so that a slab, a halo
slice and a face are CONTIGUOUS ranges of every canonical and internal array), and the halo is one
slice deep on either side because D is a one-hop stencil: M^dag M = m^2 - D_eo D_oe needs one
exchange before each D (the paper's two-deep halo trades the second exchange for redundant work).

Rank r of R owns the global slices t_lo <= t < t_lo + nt_loc (t_lo = r * Nt/R, nt_loc = Nt/R even) and
holds them, with the slice below and the slice above, as a lattice of its own with extents
(Nx, Ny, Nz, nt_loc + 2):   local slice 0 = global t_lo - 1,   1 .. nt_loc = owned,   nt_loc + 1 =
global t_lo + nt_loc   (both taken modulo Nt).  Consequences, all handled here:
  * parity: local t = global t - t_lo + 1 and t_lo is even, so (x+y+z+t) flips: GLOBAL parity p lives on
    LOCAL parity 1 - p on every rank (`local_parity`).  The staggered phases depend on x, y, z only
    (SURVEY.md C4), so they are unchanged.
  * boundary condition: the library folds its antiperiodic sign into the t-links of its own last
    slice (the upper halo, whose t-links no owned site uses) and wraps local t = nt_loc + 1 -> 0 (a hop
    no owned site makes).  The physical seam, the hop across global t = Nt-1 -> 0, is
    carried by the DATA: `local_links` negates the t-links of the global slice Nt-1 wherever it appears
    (last owned slice of the last rank, lower halo of rank 0).  Three-row link storage only: a negated
    link is not in SU(3), which two-row storage requires.
  * the owned slices are computed with qcd_dslash_range(t0 = 1, nt = nt_loc); halo slices of the
    OUTPUT are never computed, they are filled by the next exchange.

A slice of an internal vector (three colour planes, site-fastest) is three contiguous runs of
Nx/2*Ny*Nz complex numbers, 24 * Nx*Ny*Nz bytes in all: the 48 B x face sites per direction of
SURVEY.md 8(e).  `exchange_halos` moves them with torch.distributed point-to-point calls (gloo on the
CPU, nccl between GPUs); `attach` hands the library the two callbacks of its slab mode (halo fill, sum over
the ranks).  A device-initiated NVLink put fused into the stencil is the next step and is not built
(DESIGN.md section 7).
"""
from __future__ import annotations

import numpy as np


class _DevicePointer:
    """A device address dressed up for torch.as_tensor (zero-copy view of library-owned memory)."""

    def __init__(self, ptr: int, doubles: int):
        self.__cuda_array_interface__ = {"shape": (doubles,), "typestr": "<f8", "data": (ptr, False), "version": 3}


def device_view(ptr: int, doubles: int):
    import torch
    return torch.as_tensor(_DevicePointer(ptr, doubles), device="cuda")


class SlabPartition:
    """Geometry of one rank's t-slab.  dims = global (Nx, Ny, Nz, Nt)."""

    def __init__(self, dims, world: int, rank: int):
        nx, ny, nz, nt = (int(d) for d in dims)
        if world < 2:
            raise ValueError("a slab decomposition needs at least 2 ranks (1 rank: the plain path)")
        if nt % world or (nt // world) % 2 or nt // world < 2:
            raise ValueError("Nt must split into an even number (>= 2) of slices per rank")
        if not 0 <= rank < world:
            raise ValueError("rank out of range")
        self.dims, self.world, self.rank = (nx, ny, nz, nt), world, rank
        self.nt_loc = nt // world
        self.t_lo = rank * self.nt_loc
        self.local_dims = (nx, ny, nz, self.nt_loc + 2)
        self.slice_sites = nx * ny * nz             # sites of one t-slice
        self.slice_half = self.slice_sites // 2     # ... of one parity
        self.up = (rank + 1) % world                # rank that owns the slices above
        self.down = (rank - 1) % world

    # ---- parity
    @staticmethod
    def local_parity(global_parity: int) -> int:
        """Global parity p lives on local parity 1 - p (t_lo is even, the lower halo shifts t by one)."""
        return 1 - int(global_parity)

    # ---- which global slice each local slice holds
    def global_t(self) -> np.ndarray:
        """int[nt_loc + 2]: global t of local slices 0 .. nt_loc + 1."""
        return (self.t_lo - 1 + np.arange(self.nt_loc + 2)) % self.dims[3]

    # ---- canonical arrays (host side, numpy): global -> local with halos
    def local_links(self, links: np.ndarray) -> np.ndarray:
        """float64[V,4,3,3,2] global canonical links -> float64[V_loc,4,3,3,2] of the extended local
        lattice, with the antiperiodic seam folded into the t-links of the global slice Nt-1."""
        nt = self.dims[3]
        g = np.ascontiguousarray(links, dtype=np.float64).reshape(nt, self.slice_sites, 4, 3, 3, 2)
        out = g[self.global_t()].copy()
        seam = self.global_t() == nt - 1
        # the library negates the t-links of its own last slice (local seam): keep that slice's data such
        # that it is at least well defined; no owned site reads those links
        out[seam, :, 3] *= -1.0
        return out.reshape(-1, 4, 3, 3, 2)

    def local_vector(self, v: np.ndarray) -> np.ndarray:
        """float64[V/2,3,2] global canonical parity vector -> the extended local one (halos included; used
        to set up inputs and expected values -- at run time the halos come from exchange_halos)."""
        nt = self.dims[3]
        g = np.ascontiguousarray(v, dtype=np.float64).reshape(nt, self.slice_half, 3, 2)
        return np.ascontiguousarray(g[self.global_t()].reshape(-1, 3, 2))

    def owned(self, v_local: np.ndarray) -> np.ndarray:
        """The owned slices of an extended local canonical parity vector: float64[nt_loc*slice_half,3,2]."""
        return v_local.reshape(self.nt_loc + 2, self.slice_half, 3, 2)[1:-1].reshape(-1, 3, 2)

    # ---- halo exchange on an extended local vector, canonical ([t][site][3][2]) or internal ([3][t][site][2])
    def _slices(self, vec, internal: bool):
        """views (lower halo, first owned, last owned, upper halo) of a torch tensor holding one extended
        local parity vector in canonical or internal layout."""
        n = self.nt_loc
        if internal:
            a = vec.view(3, n + 2, self.slice_half * 2)
            return a[:, 0], a[:, 1], a[:, n], a[:, n + 1]
        a = vec.view(n + 2, self.slice_half * 6)
        return a[0], a[1], a[n], a[n + 1]

    def exchange_halos(self, vec, dist, internal: bool = True, staged: bool = False):
        """Fill the two halo slices of `vec` (a torch tensor, one extended local parity vector) from the
        neighbouring ranks: my first owned slice becomes the upper halo of `down`, my last owned slice
        the lower halo of `up`.  24 * Nx*Ny*Nz bytes per direction.  staged: the four slices travel through
        host copies (a CUDA vector over the gloo backend)."""
        import torch
        lo_halo, first, last, hi_halo = self._slices(vec, internal)
        send_dn, send_up = first.contiguous(), last.contiguous()
        if staged:
            send_dn, send_up = send_dn.cpu(), send_up.cpu()
        recv_lo, recv_hi = torch.empty_like(send_up), torch.empty_like(send_dn)
        ops = [dist.P2POp(dist.isend, send_up, self.up), dist.P2POp(dist.irecv, recv_lo, self.down),
               dist.P2POp(dist.isend, send_dn, self.down), dist.P2POp(dist.irecv, recv_hi, self.up)]
        for req in dist.batch_isend_irecv(ops):
            req.wait()
        lo_halo.copy_(recv_lo)
        hi_halo.copy_(recv_hi)
        return vec

    # ---- the library's slab mode (qcd_set_slab): this rank's callbacks
    def attach(self, ctx, dist, staged: bool = False):
        """Put `ctx` (a Context on the extended local lattice `local_dims`) into slab mode with callbacks
        that move the halo slices and sum the inner products over `dist`'s default group.
        staged = False: the collectives act on the device buffers themselves (backend nccl, one GPU per
        rank).  staged = True: through host copies (backend gloo; lets several ranks share ONE GPU in the
        tests -- every callback synchronises, no kernel ever waits for another rank's kernel)."""
        import torch
        vd = ctx.vector_doubles

        def lib_stream(handle):
            # the library's stream as a torch stream; handle 0 is the legacy default stream, which
            # ExternalStream(0) would NOT give (a null pointer makes torch take a fresh pool stream)
            return torch.cuda.default_stream() if not handle else torch.cuda.ExternalStream(handle)

        def halo(ptr, stream):
            vec = device_view(ptr, vd)
            with torch.cuda.stream(lib_stream(stream)):
                if staged:
                    torch.cuda.current_stream().synchronize()
                self.exchange_halos(vec, dist, internal=True, staged=staged)
                if staged:
                    torch.cuda.current_stream().synchronize()

        def allreduce(ptr, count, stream):
            buf = device_view(ptr, count)
            with torch.cuda.stream(lib_stream(stream)):
                if not staged:
                    dist.all_reduce(buf)
                    return
                torch.cuda.current_stream().synchronize()
                host = buf.cpu()
                dist.all_reduce(host)
                buf.copy_(host)
                torch.cuda.current_stream().synchronize()

        ctx.set_slab(halo, allreduce)
