"""Multi-GPU domain decomposition of the hot path: x-slabs, one rank per GPU ("MPI ... Cartesian topology",
L153 one rank per GPU).  Host-side plumbing only -- every particle and every moment is still computed
by libecpush on the rank's own GPU; this module decides who owns what and moves the two things that cross a slab face:

  * the HALO ADD of rho / Jhat / M: a slab's particles deposit on its own node planes 0..nxl-1 and on plane nxl, which is
    plane 0 of the right neighbour.  After the deposit that one plane is sent to the right neighbour, which adds it
    (moments are sums over particles, Eq. 1 / Eq. 3, so partial sums just add).  128^2 nodes x (243 + 4 nsp) doubles
    = 33 MB per face at configs[2].
  * the MIGRATION of particles whose push took them out of the slab.

How the periodic single-GPU library serves a non-periodic slab: the rank's local grid has nxl + 2 planes of cells along x:
cells 0..nxl-1 are the slab, plane nxl is the RIGHT ghost and plane nxl+1 the LEFT ghost (it is "plane -1" of the
periodic local grid).  Particles live only in the slab's cells, so their deposits reach node planes 0..nxl and nothing
wraps; a particle that leaves to the right ends in ghost plane nxl, one that leaves to the left wraps into ghost plane
nxl+1 (a particle must END in the slab or in the plane next to it; leavers() checks that by the sign of the velocity).  Local fields carry node planes 0..nxl of the slab
(plane nxl = the right neighbour's plane 0: a halo COPY the caller provides from its field solve; local_fields() cuts it
out of a global array).

Collectives: point-to-point ring exchanges (`torch.distributed` isend / irecv: NCCL on GPUs -- NVLink 5 / NVSwitch -- or
gloo on CPU tensors in the tests); sizes first, then payloads.  `LocalRing` runs all ranks of a ring in ONE process (tests
on a single GPU; no rank waits on another rank's kernel).  There is no arithmetic of the method here.
"""
from __future__ import annotations

from typing import Dict, List, Sequence, Tuple

import torch

PKEYS = ("x", "y", "z", "u", "v", "w", "q")


class SlabGrid:
    """Rank `rank` of `world` x-slabs of a periodic nx x ny x nz grid."""

    def __init__(self, nx: int, ny: int, nz: int, dx: float, dy: float, dz: float, world: int, rank: int):
        if not (0 <= rank < world) or nx < world:
            raise ValueError("need 0 <= rank < world <= nx")
        self.nx, self.ny, self.nz, self.dx, self.dy, self.dz = nx, ny, nz, dx, dy, dz
        self.world, self.rank = world, rank
        self.i0 = nx * rank // world
        self.i1 = nx * (rank + 1) // world
        self.nxl = self.i1 - self.i0
        self.left = (rank - 1) % world
        self.right = (rank + 1) % world
        self.nxl_left = nx * (self.left + 1) // world - nx * self.left // world
        self.plane = ny * nz

    # -- the local grid handed to ecsim_init_grid ----------------------------------------------------------------
    @property
    def local_dims(self) -> Tuple[int, int, int, float, float, float]:
        return (self.nxl + 2, self.ny, self.nz, self.dx, self.dy, self.dz)

    @property
    def local_nodes(self) -> int:
        return (self.nxl + 2) * self.plane

    def local_fields(self, F: torch.Tensor) -> torch.Tensor:
        """[3][global nodes] -> [3][local nodes]: node planes 0..nxl = global planes i0..i0+nxl (periodic), plane nxl+1 =
        global plane i0-1 (never gathered from: no particle sits in a ghost cell when fields are read)."""
        G = F.reshape(3, self.nx, self.plane)
        idx = [(self.i0 + l) % self.nx for l in range(self.nxl + 1)] + [(self.i0 - 1) % self.nx]
        return G[:, idx, :].reshape(3, -1).contiguous()

    # -- particles ------------------------------------------------------------------------------------------------
    def split_particles(self, part: Dict[str, torch.Tensor]) -> Dict[str, torch.Tensor]:
        """The particles of a GLOBAL set that start in this slab, in local coordinates (set-up / tests)."""
        ci = torch.clamp(torch.floor(part["x"] / self.dx), 0, self.nx - 1).to(torch.int64)
        sel = (ci >= self.i0) & (ci < self.i1)
        out = {k: part[k][sel].clone() for k in PKEYS}
        out["x"] = out["x"] - self.i0 * self.dx
        return out

    def to_global(self, part: Dict[str, torch.Tensor]) -> Dict[str, torch.Tensor]:
        out = {k: part[k].clone() for k in PKEYS}
        L = self.nx * self.dx
        x = out["x"] + self.i0 * self.dx
        out["x"] = torch.where(x >= L, x - L, x)
        return out

    def leavers(self, part: Dict[str, torch.Tensor], dt: float = None):
        """After a push on the local (periodic, nxl+2 planes) grid: masks of the particles now in the right / left ghost
        plane, and the same particles packed in the RECEIVER's local coordinates.  [7][n] tensors.

        A particle may cross several cells in a step (ECsim steps beyond the CFL limit) as long as it ENDS in the slab
        or in the plane next to it.  One that ends farther out is indistinguishable by position from another particle
        (from plane nxl-1 by +2 planes it lands in plane nxl+1, the LEFT ghost) and would be handed to the wrong
        neighbour; it is refused here instead:
          * always: the sign of the post-push velocity (x_new - x_old = dt u, Eq. 8) must agree with the side of the
            ghost plane -- this catches an end up to two planes outside the slab;
          * with `dt` given, exactly: the position the particle came from, x_new - dt u taken in the frame its class
            implies (left leavers: one period of the local grid lower), must lie in the slab."""
        x, u = part["x"], part["u"]
        ci = torch.floor(x / self.dx)
        right = ci == self.nxl
        left = ci >= self.nxl + 1
        refuse = "the slab migration exchanges with the nearest neighbours only (split the step or widen the ghost layer)"
        if bool((right & (u < 0)).any()) or bool((left & (u > 0)).any()):
            raise RuntimeError("a particle ended two cell planes outside its slab (its velocity points away from the "
                               "ghost plane it was found in): " + refuse)
        if dt is not None and x.numel():
            origin = x - dt * u - left.to(x.dtype) * ((self.nxl + 2) * self.dx)
            tol = 1e-9 * self.dx
            if bool(((origin < -tol) | (origin > self.nxl * self.dx + tol)).any()):
                raise RuntimeError("a particle ended more than one cell plane outside its slab (x_new - dt u is not "
                                   "inside the slab): " + refuse)
        stay = ~(right | left)
        pack_r = torch.stack([part[k][right] for k in PKEYS])
        pack_l = torch.stack([part[k][left] for k in PKEYS])
        # receiver frames: right neighbour starts at our i1; left neighbour's slab ends at our i0
        pack_r[0] = pack_r[0] - self.nxl * self.dx
        pack_l[0] = pack_l[0] - (self.nxl + 2) * self.dx + self.nxl_left * self.dx
        return stay, pack_r, pack_l

    def merge(self, part: Dict[str, torch.Tensor], stay: torch.Tensor, from_left: torch.Tensor,
              from_right: torch.Tensor) -> Dict[str, torch.Tensor]:
        """The slab's particles after the exchange: those that stayed + the arrivals (unsorted: load with sorted = 0)."""
        out = {}
        for i, k in enumerate(PKEYS):
            out[k] = torch.cat([part[k][stay], from_left[i], from_right[i]]).contiguous()
        x = out["x"]
        if x.numel() and not bool(((x >= 0) & (x < self.nxl * self.dx)).all()):
            raise RuntimeError("a particle moved more than one cell plane in one step: slab migration needs |dx| < cell")
        return out

    # -- moments --------------------------------------------------------------------------------------------------
    def halo_planes(self, rho: torch.Tensor, J: torch.Tensor, M: torch.Tensor) -> torch.Tensor:
        """The right-halo node plane (local plane nxl) of rho [nsp][nodes_l], J [nsp][3][nodes_l], M [nodes_l][K] packed
        into one contiguous buffer for the right neighbour; the plane is zeroed locally (it is not ours)."""
        nsp = rho.shape[0]
        p0, p1 = self.nxl * self.plane, (self.nxl + 1) * self.plane
        r = rho.reshape(nsp, -1)[:, p0:p1]
        j = J.reshape(nsp, 3, -1)[:, :, p0:p1]
        m = M.reshape(self.local_nodes, -1)[p0:p1]
        buf = torch.cat([r.reshape(-1), j.reshape(-1), m.reshape(-1)]).contiguous()
        r.zero_(); j.zero_(); m.zero_()
        return buf

    def add_halo(self, buf: torch.Tensor, rho: torch.Tensor, J: torch.Tensor, M: torch.Tensor):
        """Add the left neighbour's halo plane onto our node plane 0."""
        nsp = rho.shape[0]
        P = self.plane
        K = M.reshape(self.local_nodes, -1).shape[1]
        o = 0
        rho.reshape(nsp, -1)[:, :P] += buf[o:o + nsp * P].reshape(nsp, P); o += nsp * P
        J.reshape(nsp, 3, -1)[:, :, :P] += buf[o:o + 3 * nsp * P].reshape(nsp, 3, P); o += 3 * nsp * P
        M.reshape(self.local_nodes, -1)[:P] += buf[o:o + P * K].reshape(P, K)

    def owned(self, a: torch.Tensor, node_axis: int) -> torch.Tensor:
        """The owned node planes 0..nxl-1 of a local array whose axis `node_axis` runs over local nodes."""
        return a.narrow(node_axis, 0, self.nxl * self.plane)


# ---------------------------------------------------------------------------------------------------------------------
class DistRing:
    """Ring exchange over torch.distributed (backend nccl for CUDA tensors, gloo for CPU tensors)."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist = dist
        self.group = group
        self.rank = dist.get_rank(group)
        self.world = dist.get_world_size(group)
        self.left = (self.rank - 1) % self.world
        self.right = (self.rank + 1) % self.world

    def _sendrecv(self, send: torch.Tensor, dst: int, recv: torch.Tensor, src: int):
        if self.world == 1:
            recv.copy_(send)
            return
        ops = [self.dist.P2POp(self.dist.isend, send, dst, self.group), self.dist.P2POp(self.dist.irecv, recv, src, self.group)]
        for r in self.dist.batch_isend_irecv(ops):
            r.wait()

    def shift_right(self, buf: torch.Tensor) -> torch.Tensor:
        """Fixed-size buffer to the right neighbour; returns what the left neighbour sent."""
        out = torch.empty_like(buf)
        self._sendrecv(buf, self.right, out, self.left)
        return out

    def exchange(self, to_right: torch.Tensor, to_left: torch.Tensor) -> Tuple[torch.Tensor, torch.Tensor]:
        """Variable-size [7][n] packs both ways: (from_left, from_right).  Sizes travel first."""
        dev = to_right.device
        nr = torch.tensor([to_right.shape[1]], dtype=torch.int64, device=dev)
        nl = torch.tensor([to_left.shape[1]], dtype=torch.int64, device=dev)
        from_left_n = torch.empty_like(nr)
        from_right_n = torch.empty_like(nl)
        self._sendrecv(nr, self.right, from_left_n, self.left)
        self._sendrecv(nl, self.left, from_right_n, self.right)
        from_left = torch.empty(7, int(from_left_n), dtype=to_right.dtype, device=dev)
        from_right = torch.empty(7, int(from_right_n), dtype=to_left.dtype, device=dev)
        self._sendrecv(to_right.contiguous(), self.right, from_left, self.left)
        self._sendrecv(to_left.contiguous(), self.left, from_right, self.right)
        return from_left, from_right


class LocalRing:
    """All ranks of a ring in one process: the same two exchanges on lists indexed by rank (single-GPU tests)."""

    def __init__(self, world: int):
        self.world = world

    def shift_right(self, bufs: Sequence[torch.Tensor]) -> List[torch.Tensor]:
        return [bufs[(r - 1) % self.world].clone() for r in range(self.world)]

    def exchange(self, to_right: Sequence[torch.Tensor], to_left: Sequence[torch.Tensor]):
        from_left = [to_right[(r - 1) % self.world].clone() for r in range(self.world)]
        from_right = [to_left[(r + 1) % self.world].clone() for r in range(self.world)]
        return from_left, from_right
