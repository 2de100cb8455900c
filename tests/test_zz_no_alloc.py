"""sldg_density_static: the density for callers that cannot allocate device memory.

Some users of the library need rho at a point where they may not call cudaMalloc: an application whose own pool already
holds all of HBM (a new allocation fails or shrinks the pool), a loop that cannot take the device-wide synchronisation of
cudaMalloc / cudaFree, a plug-in that works on pointers lent by its host.  sldg_density is out of reach for them (its context
allocates tables and it wants a workspace), so the library has one context-free entry point whose partial sums sit in a fixed
8 MiB array inside the library image.  This file checks that entry point against the ordinary sldg_density path:

  * the same rho, at the per-operation bar the other GPU tests use (1e-12 relative to max|rho|), for fp64 and fp32 fields,
    2-wide and scalar load paths, one and several v chunks;
  * on calls IN A ROW that share the fixed array: a large problem, then a smaller one whose partial sums land on top of the
    first call's left-overs, then the first again; the array is never cleared, so a stage that read a stale partial sum would
    show here; repeated calls give the same bits;
  * a grid beyond the fixed array's capacity is refused with SLDG_ETOOLARGE and its message, bad arguments with SLDG_EINVAL,
    and neither touches the device.

The file is named test_zz_* so that pytest collects it last: `pytest -x` stops at the first failure, and a failure here must
not hide the parity tests.  It needs nothing from the tests before it and runs alone in a fresh process as well.
"""
import ctypes as C

import numpy as np
import pytest
import torch

import workloads as W

pytestmark = pytest.mark.gpu

TOL_SWEEP = 1e-12          # the bar of tests/test_gpu_parity.py for one operation


@pytest.fixture(scope="module")
def P():
    import paper_2110_14557_b200 as pkg
    if not torch.cuda.is_available():
        pytest.fail("gpu test without a CUDA device")
    return pkg


def default_domain(dx, dv):
    dom = []
    for a in range(dx + dv):
        dom += [0.0, 1.0 + a] if a < dx else [-2.0 - a, 2.0 + a]
    return dom


def velocity_weights(P, dx, dv, cells, k, dom):
    """Wv[v] = prod_d h_{v_d} w_{j_d}, v_1 fastest: what a caller of sldg_density_static builds once on the host
    (w = the library's Gauss-Legendre weights on [0,1])."""
    _, w = P.gauss_legendre(k)
    Wv = np.ones(1)
    for a in range(dx, dx + dv):
        h = (dom[2 * a + 1] - dom[2 * a]) / cells[a]
        wa = np.tile(h * w, cells[a])                      # node n = i (k+1) + j  ->  h w_j
        Wv = (wa[:, None] * Wv[None, :]).reshape(-1)       # the new axis is slower than the ones before it
    return torch.from_numpy(np.ascontiguousarray(Wv)).cuda()


class Case:
    """One geometry: a context for the existing path, a seeded field, the caller-side weights, and the existing path's rho."""

    def __init__(self, P, dx, dv, cells, k, prec, seed):
        dom = default_domain(dx, dv)
        self.g = P.Sldg(dx, dv, cells, k, dom, precision=prec)
        f = W.random_field(self.g.shape, seed=seed)
        if prec == "f32":
            f = f.to(torch.float32)
        self.f = f.to(self.g.device).contiguous()
        self.Wv = velocity_weights(P, dx, dv, cells, k, dom)
        assert self.Wv.numel() * self.g.X == self.f.numel()
        self.want = self.g.density(self.f).reshape(-1).cpu().numpy()
        self.rho = torch.empty(self.g.X, dtype=torch.float64, device=self.g.device)      # the caller's output buffer

    def run(self, P):
        self.rho.fill_(float("nan"))                                                     # every entry must be written
        P.density_static(self.f, self.Wv, rho=self.rho)
        return self.rho.cpu().numpy()


def rel_inf(g, o):
    return float(np.abs(g - o).max() / np.abs(o).max())


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_static_density_equals_the_context_path_on_calls_in_a_row(P, prec):
    big = Case(P, 2, 2, [32, 32, 16, 16], 1, prec, seed=41)        # X = 4096 (2-wide loads), V = 1024: several v chunks
    small = Case(P, 2, 2, [7, 5, 6, 9], 2, prec, seed=42)          # X = 315, odd: scalar loads, ragged last tile
    six = Case(P, 3, 3, [4, 3, 5, 3, 4, 2], 1, prec, seed=43)      # 3x3v layout, X = 480, V = 192
    first = big.run(P)
    assert rel_inf(first, big.want) <= TOL_SWEEP
    # second call straight after the first: its partial sums overwrite part of what the first call left in the fixed array
    assert rel_inf(small.run(P), small.want) <= TOL_SWEEP
    assert rel_inf(six.run(P), six.want) <= TOL_SWEEP
    # and back: same input, same bits as before the other problems used the array
    again = big.run(P)
    assert np.array_equal(first, again)
    assert np.array_equal(big.run(P), again)
    assert np.isfinite(again).all()


def test_static_density_of_a_constant_is_the_velocity_volume(P):
    """A check that does not go through the other path: f = 1 integrates to the volume of the velocity box."""
    dx, dv, cells, k = 2, 3, [6, 4, 5, 4, 3], 1
    dom = default_domain(dx, dv)
    Wv = velocity_weights(P, dx, dv, cells, k, dom)
    X = (cells[0] * (k + 1)) * (cells[1] * (k + 1))
    f = torch.ones(Wv.numel() * X, dtype=torch.float64, device="cuda")
    vol = np.prod([dom[2 * a + 1] - dom[2 * a] for a in range(dx, dx + dv)])
    for _ in range(2):
        rho = P.density_static(f, Wv).cpu().numpy()
        assert rho.shape == (X,) and np.abs(rho - vol).max() <= 1e-13 * vol


def test_static_density_refuses_what_its_fixed_array_cannot_hold(P):
    L = P.lib()
    cap = P.density_static_max_x()
    assert cap == 1 << 20
    buf = torch.zeros(64, dtype=torch.float64, device="cuda")
    p = C.c_void_p(buf.data_ptr())
    err = C.c_int(7)
    # one x node too many: refused before any launch (the pointers are never dereferenced)
    rc = L.sldg_density_static(p, p, cap + 1, 4, 0, p, None, C.byref(err))
    assert rc == -5 and err.value == 0
    assert b"SLDG_DENSITY_STATIC_MAX_X" in L.sldg_strerror(rc)
    # bad arguments
    assert L.sldg_density_static(None, p, 8, 4, 0, p, None, None) == -1
    assert L.sldg_density_static(p, None, 8, 4, 0, p, None, None) == -1
    assert L.sldg_density_static(p, p, 8, 4, 0, None, None, None) == -1
    assert L.sldg_density_static(p, p, 0, 4, 0, p, None, None) == -1
    assert L.sldg_density_static(p, p, 8, 0, 0, p, None, None) == -1
    assert L.sldg_density_static(p, p, 8, 4, 2, p, None, None) == -1
    torch.cuda.synchronize()
    # the device is still healthy and the entry point still works
    Wv = torch.full((4,), 0.5, dtype=torch.float64, device="cuda")
    f = torch.arange(32, dtype=torch.float64, device="cuda")
    rho = P.density_static(f, Wv).cpu().numpy()
    assert np.array_equal(rho, 0.5 * f.cpu().numpy().reshape(4, 8).sum(axis=0))
