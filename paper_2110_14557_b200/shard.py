"""v-axis domain decomposition of a Strang step over ranks ("Communication", Fig. 3; PAPER.md:137-141;
SURVEY 8(f) rank 4 tail).  HOST-SIDE PLUMBING ONLY: which slab a rank owns, how wide its halo is, what is exchanged and
reduced.  Every arithmetic step stays in the engine the caller supplies (the CUDA context `Sldg` on a GPU; the tests
drive the same plumbing over CPU buffers with gloo).  BASELINE.json fixes ONE GPU for this build ("replicas only",
DESIGN.md section 9), so nothing in bench.py uses this module; it is the design of the next row, kept testable.

Decomposition.  The SLOWEST velocity axis (axis d-1) is cut into `world` contiguous slabs of n_loc cells (slabs differ by at
most one cell when the cell count is not a multiple of `world`; `start` is a slab's first cell).  A rank stores
its slab plus H halo cells on either side, f_ext = [n_loc + 2H cells of v_last][...all other axes...], i.e. one contiguous
array in the library's layout whose last axis has n_loc + 2H cells and whose domain on that axis is widened by H cells.

  * x sweeps: the shift of a line depends on ITS velocity node only -> purely local; a context created
    on the widened sub-domain builds the right tables for the slab's own nodes (the halo cells are swept too: harmless).
  * rho: a rank sums its INTERIOR cells (the interior is a contiguous sub-array of f_ext, handed to a context of the
    interior geometry), then ONE all-reduce of X doubles (<= 0.9 MB for the BASELINE configs); every rank solves the
    Poisson problem redundantly (the field solve is tiny).
  * v sweeps along axes below the cut: local.  The sweep along the cut axis reads cells i-s and i-s-1 (eq. (3)): with
    |delta| <= H - 1 cells the interior depends on the slab plus H cells of either neighbour.  The halos are exchanged once
    per step, after the first x half step (the paper exchanges one-sidedly per sign of the shift; here both sides are
    filled because the sign changes with the x node).  The sweep then runs as the library's PERIODIC sweep on the
    widened array: the wrap-around only pollutes halo cells, which are overwritten by the next exchange.
  * dim_v > dim_x (2x3v): the cut axis is not advected (reading D): H = 0, no halo traffic at all.

The result on the interiors equals the single-domain step up to the summation order of rho (all-reduce of per-rank
partial sums instead of one sum): 1e-15 relative, far inside the parity bars.
"""
import math


class Geometry:
    """cells / domain of a problem in the library's convention (x axes first)."""

    def __init__(self, dim_x, dim_v, cells, degree, domain):
        self.dim_x, self.dim_v, self.degree = int(dim_x), int(dim_v), int(degree)
        self.cells = [int(c) for c in cells]
        self.domain = [float(v) for v in domain]
        self.d = self.dim_x + self.dim_v

    def with_last_axis(self, ncells, lo, hi):
        cells = self.cells[:-1] + [int(ncells)]
        domain = self.domain[:-2] + [float(lo), float(hi)]
        return Geometry(self.dim_x, self.dim_v, cells, self.degree, domain)


def halo_cells(geom, e_max, dt):
    """Halo width in cells for fields with |E_d| <= e_max on the cut axis: |delta| = e_max dt / h_v, donors i-s, i-s-1
    -> ceil(|delta|) + 1 cells; 0 when the cut axis is not advected (dim_v > dim_x)."""
    if geom.dim_v > geom.dim_x:
        return 0
    lo, hi = geom.domain[-2], geom.domain[-1]
    h = (hi - lo) / geom.cells[-1]
    return int(math.ceil(abs(e_max) * abs(dt) / h)) + 1


class HaloTooNarrow(RuntimeError):
    pass


def cuda_interior_density(P, interior):
    """-> callable(f_interior) for VShard(interior_density=...): rho of the interior slab through sldg_density_static, which
    takes the slab (a contiguous sub-array of the extended array) and its velocity weights and needs neither a context nor a
    workspace.  P is the binding module (paper_2110_14557_b200); the weights prod_d h_{v_d} w_{j_d} of the INTERIOR geometry
    are built here once, on the host, and uploaded."""
    import numpy as np
    import torch
    _, w = P.gauss_legendre(interior.degree)
    Wv = np.ones(1)
    for a in range(interior.dim_x, interior.d):
        h = (interior.domain[2 * a + 1] - interior.domain[2 * a]) / interior.cells[a]
        Wv = (np.tile(h * w, interior.cells[a])[:, None] * Wv[None, :]).reshape(-1)
    Wv_dev = torch.from_numpy(np.ascontiguousarray(Wv)).cuda()
    k1 = interior.degree + 1
    xshape = tuple(reversed([c * k1 for c in interior.cells[:interior.dim_x]]))

    def density(f_int):
        return P.density_static(f_int, Wv_dev).reshape(xshape)
    return density


class VShard:
    """One rank's share of a v-sharded problem.

    make_engine(geometry) -> object with advect_x(f, tau), advect_v(f, E, tau), density(f) -> rho, poisson(rho) -> E acting
    on arrays of that geometry in place / by value (the CUDA binding's `Sldg` has exactly these calls).
    `dist` is torch.distributed (already initialised) or None for a single rank.
    `interior_density` (optional): callable(f_interior) -> rho of the rank's interior cells.  Without it a SECOND engine is
    built on the interior geometry just for rho; with the CUDA binding that engine is a full context whose workspace holds
    another |f_interior| values of device memory.  `cuda_interior_density` below gives the CUDA path a density that needs no
    context and no workspace (sldg_density_static), so the rank carries one workspace only."""

    def __init__(self, geom, rank, world, halo, make_engine, dist=None, interior_density=None):
        n = geom.cells[-1]
        self.geom, self.rank, self.world, self.H, self.dist = geom, int(rank), int(world), int(halo), dist
        if not 0 <= self.rank < self.world or self.world > n:
            raise ValueError(f"{world} ranks for {n} cells on the cut axis")
        # Slabs need not be equal: the first n % world ranks own one cell more (20 cells of cfg4/cfg5 over 8 ranks: 3,3,3,3,2,2,2,2).
        # Nothing else depends on equal slabs -- a halo is H cells whatever the neighbour's size, rho is an all-reduce.
        q, rem = divmod(n, self.world)
        self.n_loc = q + (1 if self.rank < rem else 0)
        self.start = self.rank * q + min(self.rank, rem)          # first cell of the slab on the cut axis
        if self.H > q:
            raise ValueError("halo wider than the smallest slab: use fewer ranks or a smaller time step")
        lo, hi = geom.domain[-2], geom.domain[-1]
        h = (hi - lo) / n
        a = lo + self.start * h
        b = lo + (self.start + self.n_loc) * h
        self.interior = geom.with_last_axis(self.n_loc, a, b)
        self.extended = geom.with_last_axis(self.n_loc + 2 * self.H, a - self.H * h, b + self.H * h)
        self.eng_ext = make_engine(self.extended)
        self.interior_density = interior_density
        self.eng_int = None if interior_density is not None else (make_engine(self.interior) if self.H else self.eng_ext)
        self.k1 = geom.degree + 1
        self.h_cut = h

    # ---- views of the extended array (axis 0 of the array = slowest axis = the cut axis, in nodes)
    def interior_of(self, f_ext):
        r = self.H * self.k1
        return f_ext[r:f_ext.shape[0] - r] if r else f_ext

    def exchange_halos(self, f_ext):
        """Fill the H halo cells on either side from the neighbouring ranks' interiors (periodic ring)."""
        if not self.H:
            return
        import torch
        r = self.H * self.k1
        top = f_ext[f_ext.shape[0] - 2 * r:f_ext.shape[0] - r].contiguous()      # my last H interior cells -> next rank's lower halo
        bot = f_ext[r:2 * r].contiguous()                                        # my first H interior cells -> previous rank's upper halo
        if self.world == 1 or self.dist is None:
            f_ext[:r].copy_(top)
            f_ext[f_ext.shape[0] - r:].copy_(bot)
            return
        nxt, prv = (self.rank + 1) % self.world, (self.rank - 1) % self.world
        lower, upper = torch.empty_like(top), torch.empty_like(bot)
        ops = [self.dist.P2POp(self.dist.isend, top, nxt, tag=1), self.dist.P2POp(self.dist.irecv, lower, prv, tag=1),
               self.dist.P2POp(self.dist.isend, bot, prv, tag=2), self.dist.P2POp(self.dist.irecv, upper, nxt, tag=2)]
        for w in self.dist.batch_isend_irecv(ops):
            w.wait()
        f_ext[:r].copy_(lower)
        f_ext[f_ext.shape[0] - r:].copy_(upper)

    def density(self, f_ext):
        """rho of the WHOLE problem: the rank's interior partial sum, all-reduced."""
        f_int = self.interior_of(f_ext)
        rho = self.interior_density(f_int) if self.interior_density is not None else self.eng_int.density(f_int)
        if self.world > 1 and self.dist is not None:
            self.dist.all_reduce(rho, op=self.dist.ReduceOp.SUM)
        return rho

    def check_halo(self, E, dt):
        """The halo width was fixed at construction from an estimate of max|E|.  If the field has grown past it (two-stream
        runs do), donors of interior cells would come from the periodic wrap of the widened slab: silently wrong.  So the
        cut-axis component of the field just solved (X doubles, identical on every rank) is checked every step; the read-back
        of its maximum synchronises the stream once per step."""
        if not self.H:
            return
        emax = float(abs(E[-1]).max())
        need = int(math.ceil(emax * abs(dt) / self.h_cut)) + 1
        if need > self.H:
            raise HaloTooNarrow(f"max|E| = {emax:.6g} on the cut axis needs a halo of {need} cells for dt = {dt:g}, "
                                f"this shard was built with {self.H}: rebuild it with halo_cells(geom, e_max, dt) for a larger e_max")

    def step(self, f_ext, dt):
        """One Strang step on this rank's extended slab; returns (rho, E) of the step."""
        self.eng_ext.advect_x(f_ext, dt / 2.0)
        rho = self.density(f_ext)
        E = self.eng_ext.poisson(rho)                      # redundant on every rank
        self.check_halo(E, dt)
        self.exchange_halos(f_ext)
        self.eng_ext.advect_v(f_ext, E, dt)
        self.eng_ext.advect_x(f_ext, dt / 2.0)
        return rho, E
