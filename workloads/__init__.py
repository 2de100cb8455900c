"""Seeded, synthetic input generators shared by the tests, bench.py and smoke().

This module holds NONE of the method's arithmetic: no Gauss-Legendre nodes, no A/B
matrices, no sweeps.  It only (a) names the five BASELINE.json configurations,
(b) evaluates the analytic initial data f0 at node coordinates that the CALLER
supplies (each side -- oracle or CUDA library -- computes its own coordinates), and
(c) draws seeded random fields / shift tables.  Arrays are torch tensors (float64) so
that the same generator fills a 2 MB CPU array for the oracle and a 10.9 GB device
array for bench.py without a host round trip.

Array convention: flat index n = n_0 + D_0 (n_1 + D_1 (...)),
axis order x_1..x_dx, v_1..v_dv, x_1 fastest.  As a torch tensor the shape is
(D_{d-1}, ..., D_1, D_0).

The Landau data follow the paper (alpha=0.01, k=0.5,
[0,4pi]^dx x [-6,6]^dv); the two-stream data are BASELINE.json's (not in the paper);
the bump-on-tail data are the paper's second validation case.
No dataset or benchmark suite is involved.
"""
import math

import torch

SEED = 211014557

_PI = math.pi

CONFIGS = [
    dict(name="cfg1_4d_landau_8x16_k1", dim_x=2, dim_v=2, cells=[8, 8, 16, 16], degree=1,
         domain=[0, 4 * _PI, 0, 4 * _PI, -6, 6, -6, 6], dt=0.1, steps=10, ic="landau",
         ic_args=dict(eps=0.01, k=0.5, axes=[0, 1])),
    dict(name="cfg2_4d_twostream_64x64_k2", dim_x=2, dim_v=2, cells=[64, 64, 64, 64], degree=2,
         domain=[0, 10 * _PI, 0, 10 * _PI, -6, 6, -6, 6], dt=0.05, steps=10, ic="two_stream",
         ic_args=dict(eps=1e-3, k=0.2, v0=2.4)),
    dict(name="cfg3_5d_landau_32x32_k1", dim_x=2, dim_v=3, cells=[32, 32, 32, 32, 32], degree=1,
         domain=[0, 4 * _PI, 0, 4 * _PI, -6, 6, -6, 6, -6, 6], dt=0.1, steps=10, ic="landau",
         ic_args=dict(eps=0.01, k=0.5, axes=[0])),
    dict(name="cfg4_6d_landau_20x20_k1", dim_x=3, dim_v=3, cells=[20] * 6, degree=1,
         domain=[0, 4 * _PI] * 3 + [-6, 6] * 3, dt=0.1, steps=10, ic="landau",
         ic_args=dict(eps=0.01, k=0.5, axes=[0, 1, 2])),
    dict(name="cfg5_6d_twostream_24x20_k1", dim_x=3, dim_v=3, cells=[24, 24, 24, 20, 20, 20], degree=1,
         domain=[0, 10 * _PI] * 3 + [-6, 6] * 3, dt=0.05, steps=10, ic="two_stream",
         ic_args=dict(eps=1e-3, k=0.2, v0=2.4)),
]

# the paper's own second validation case (bump-on-tail, on
# [0,20pi/3]^dx x [-9,9]^dv, 4th order = degree 3, time step 0.1) and CFL > 1 time steps.
# The paper ran 144^5 / 72^6 degrees of freedom on 32 / 64 GPUs; these are sized for one B200.
_L = 20 * _PI / 3
NEXT_CONFIGS = [
    dict(name="bot_4d_k3_small", dim_x=2, dim_v=2, cells=[6, 5, 8, 7], degree=3,
         domain=[0, _L, 0, _L, -9, 9, -9, 9], dt=0.1, steps=10, ic="bump_on_tail",
         ic_args=dict(eps=0.03, k=0.3)),
    dict(name="bot_5d_k3_16", dim_x=2, dim_v=3, cells=[16] * 5, degree=3,
         domain=[0, _L, 0, _L, -9, 9, -9, 9, -9, 9], dt=0.1, steps=10, ic="bump_on_tail",
         ic_args=dict(eps=0.03, k=0.3)),
    dict(name="bot_6d_k3_9", dim_x=3, dim_v=3, cells=[9] * 6, degree=3,
         domain=[0, _L] * 3 + [-9, 9] * 3, dt=0.1, steps=10, ic="bump_on_tail",
         ic_args=dict(eps=0.03, k=0.3)),
]


def with_cfl(cfg, cfl):
    """Same problem with the time step chosen so that the largest x shift max|v| (dt/2) / h_x is `cfl` cells
    (PAPER.md:351-357 runs CFL 1..5)."""
    out = dict(cfg)
    dx = cfg["dim_x"]
    vmax = max(abs(b) for b in cfg["domain"][2 * dx:])
    hx = min((cfg["domain"][2 * a + 1] - cfg["domain"][2 * a]) / cfg["cells"][a] for a in range(dx))
    out["dt"] = 2.0 * cfl * hx / vmax
    out["name"] = cfg["name"] + f"_cfl{cfl:g}"
    return out


def scaled(cfg, cells):
    """Same dimensions, degree, domain, dt and initial data; fewer cells (a 'scaled replica')."""
    out = dict(cfg)
    out["cells"] = [int(c) for c in cells]
    out["name"] = cfg["name"] + "_scaled_" + "x".join(str(c) for c in out["cells"])
    return out


def field_shape(cfg):
    k1 = cfg["degree"] + 1
    return tuple(c * k1 for c in reversed(cfg["cells"]))


def field_elems(cfg):
    n = 1
    for s in field_shape(cfg):
        n *= s
    return n


def _as_tensors(coords, device):
    return [torch.as_tensor(c, dtype=torch.float64, device=device) for c in coords]


def _outer_x_first(factors):
    """factors[a] is a 1-D tensor over axis a.  Returns prod_a factors[a][n_a] with shape
    (D_{m-1}, ..., D_0) (axis 0 last/fastest)."""
    m = len(factors)
    out = None
    for a, fa in enumerate(factors):
        shp = [1] * m
        shp[m - 1 - a] = fa.numel()
        t = fa.reshape(shp)
        out = t if out is None else out * t
    return out


def initial_data(cfg, coords, device="cpu", out=None):
    """f0 of `cfg` at the tensor-product nodes.  coords[a] = node coordinates of axis a
    (length D_a), supplied by the caller.  Returns a float64 tensor of shape field_shape(cfg)."""
    dx, dv = cfg["dim_x"], cfg["dim_v"]
    c = _as_tensors(coords, device)
    assert len(c) == dx + dv
    xs, vs = c[:dx], c[dx:]
    a = cfg["ic_args"]
    xshape = tuple(t.numel() for t in reversed(xs))
    # spatial factor 1 + eps * sum_j cos(k x_j)
    X = torch.ones(xshape, dtype=torch.float64, device=device)
    if cfg["ic"] == "landau":
        for j in a["axes"]:
            f = [torch.ones_like(t) for t in xs]
            f[j] = torch.cos(a["k"] * xs[j])
            X = X + a["eps"] * _outer_x_first(f)
        V = _outer_x_first([torch.exp(-0.5 * t * t) for t in vs]) / (2 * _PI) ** (dv / 2)
    elif cfg["ic"] == "two_stream":
        f = [torch.ones_like(t) for t in xs]
        f[0] = torch.cos(a["k"] * xs[0])
        X = X + a["eps"] * _outer_x_first(f)
        g1 = torch.exp(-0.5 * (vs[0] - a["v0"]) ** 2) + torch.exp(-0.5 * (vs[0] + a["v0"]) ** 2)
        V = _outer_x_first([g1] + [torch.exp(-0.5 * t * t) for t in vs[1:]]) / (2 * (2 * _PI) ** (dv / 2))
    elif cfg["ic"] == "bump_on_tail":
        # (0.9 exp(-v1^2/2) + 0.2 exp(-2 (v1-4.5)^2)) exp(-sum_{i>=2} v_i^2/2) / (2 pi)^{dv/2}
        #               * (1 + 0.03 sum_i cos(0.3 x_i))
        for j in range(dx):
            f = [torch.ones_like(t) for t in xs]
            f[j] = torch.cos(a["k"] * xs[j])
            X = X + a["eps"] * _outer_x_first(f)
        g1 = 0.9 * torch.exp(-0.5 * vs[0] ** 2) + 0.2 * torch.exp(-2.0 * (vs[0] - 4.5) ** 2)
        V = _outer_x_first([g1] + [torch.exp(-0.5 * t * t) for t in vs[1:]]) / (2 * _PI) ** (dv / 2)
    else:
        raise ValueError(cfg["ic"])
    Vb = V.reshape(tuple(V.shape) + (1,) * dx)
    Xb = X.reshape((1,) * dv + tuple(X.shape))
    if out is None:
        return Vb * Xb
    return torch.mul(Vb, Xb, out=out)


def generator(seed=SEED, device="cpu"):
    g = torch.Generator(device=device)
    g.manual_seed(int(seed))
    return g


def random_field(shape, seed=SEED, kind="uniform", base=None, device="cpu"):
    """kind='uniform': U(0,1);  kind='perturbed': base * (1 + 1e-3 U(-1,1))."""
    g = generator(seed, device)
    u = torch.rand(tuple(shape), dtype=torch.float64, device=device, generator=g)
    if kind == "uniform":
        return u
    if kind == "perturbed":
        return base * (1.0 + 1e-3 * (2.0 * u - 1.0))
    raise ValueError(kind)


def perturb_inplace(f, seed=SEED, amplitude=1e-3, slab_elems=1 << 27):
    """f *= 1 + amplitude * U(-1,1), slab by slab along the slowest axis (no |f|-sized temporary: usable on a
    57 GB device array).  The draw depends on the slab size, so callers that compare must share it."""
    g = generator(seed, f.device)
    flat = f.view(-1)
    n = flat.numel()
    for a in range(0, n, slab_elems):
        b = min(n, a + slab_elems)
        u = torch.rand(b - a, dtype=torch.float64, device=f.device, generator=g)
        flat[a:b].mul_(1.0 + amplitude * (2.0 * u - 1.0))
    return f


def delta_table(n, kind, seed=SEED, ncells=None):
    """Shift tables (in cells) for the single-sweep test hook; returns float64 CPU tensor of length n.
      'int0', 'int+1', 'int-1', 'int+3', 'int-3', 'intwrap' (= ncells+2), 'intmix' (seeded integers in [-6,6])
      'cfl'   : U(-5.5, 5.5)   (CFL > 1)
      'small' : U(-1, 1)       (the BASELINE.json regime |delta| < 1)
      'edge'  : values at +-1e-12 and 1 -+ 1e-12 around integers, cycled
    """
    g = generator(seed)
    if kind.startswith("int") and kind not in ("intwrap", "intmix"):
        return torch.full((n,), float(int(kind[3:])), dtype=torch.float64)
    if kind == "intwrap":
        return torch.full((n,), float(ncells + 2), dtype=torch.float64)
    if kind == "intmix":
        return torch.randint(-6, 7, (n,), generator=g).to(torch.float64)
    if kind == "cfl":
        return (torch.rand(n, dtype=torch.float64, generator=g) * 2 - 1) * 5.5
    if kind == "small":
        return torch.rand(n, dtype=torch.float64, generator=g) * 2 - 1
    if kind == "edge":
        vals = torch.tensor([1e-12, -1e-12, 1 - 1e-12, -1 + 1e-12, 2 + 1e-12, -3 - 1e-12, 0.5, -0.5],
                            dtype=torch.float64)
        return vals[torch.arange(n) % vals.numel()].clone()
    raise ValueError(kind)


def random_E(dim_x, xshape, seed=SEED, amplitude=1.0, device="cpu"):
    """Seeded electric field [dim_x, *xshape], U(-amplitude, amplitude)."""
    g = generator(seed, device)
    u = torch.rand((dim_x,) + tuple(xshape), dtype=torch.float64, device=device, generator=g)
    return amplitude * (2.0 * u - 1.0)
