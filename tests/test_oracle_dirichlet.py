"""Pins of the oracle's conducting-pipe Poisson solver (the paper's own: eqs. 15-27).
Geometry reading (N1): wall = node 0 and the virtual node n one spacing beyond the last
stored node, so m = n-1 interior nodes per axis and 2(m+1) = 2n points in the odd extension (eq. 18)."""
import numpy as np
import pytest
import scipy.sparse as sp
import scipy.sparse.linalg as spla

from workloads import make_grid


def pipe_grid(nx, ny, half_x, half_y):
    g = make_grid(nx, half_x, ny=ny, half_y=half_y)
    g["boundary"] = 1
    return g


def spacing(g):
    return (g["xmax"] - g["xmin"]) / (g["nx"] - 1), (g["ymax"] - g["ymin"]) / (g["ny"] - 1)


def test_dirichlet_equals_sparse_direct_solve_of_eq17(orc):
    """eq. 17 with u = 0 on the wall, solved directly (scipy sparse LU) on a 16 x 8 grid with dx != dy and a
    random source: the FFT route of eqs. 18-27 must give the same interior potential."""
    nx, ny = 16, 8
    g = pipe_grid(nx, ny, 0.03, 0.011)
    dx, dy = spacing(g)
    rng = np.random.Generator(np.random.PCG64(11))
    Q = rng.random((ny, nx))
    n_total = 37.0
    u = orc.poisson(Q, g, n_total)
    mx, my = nx - 1, ny - 1                                   # interior nodes 1..n-1
    def lap1(m, d):
        return sp.diags([np.ones(m - 1), -2.0 * np.ones(m), np.ones(m - 1)], [-1, 0, 1]) / d ** 2
    A = sp.kron(sp.identity(my), lap1(mx, dx)) + sp.kron(lap1(my, dy), sp.identity(mx))
    f = Q[1:, 1:] / (n_total * dx * dy)
    want = spla.spsolve(sp.csc_matrix(A), -f.ravel()).reshape(my, mx)       # laplace(u) = -f  (A4)
    assert np.abs(u[1:, 1:] - want).max() < 1e-12 * np.abs(want).max()
    assert np.all(u[0, :] == 0.0) or np.abs(u[0, :]).max() < 1e-15 * np.abs(want).max()   # wall row / column
    assert np.abs(u[:, 0]).max() < 1e-15 * np.abs(want).max()


@pytest.mark.parametrize("a,b", [(1, 1), (3, 2), (7, 5)])
def test_dirichlet_sine_eigenfunction(orc, a, b):
    """sin(pi a i/n) sin(pi b j/n) is an eigenvector of the five-point Laplacian with Dirichlet walls at 0 and n:
    eigenvalue -4 (sin^2(pi a/2n)/dx^2 + sin^2(pi b/2n)/dy^2) -- the symbol of eq. 25 at (p, q) = (a, b)."""
    nx, ny = 32, 16
    g = pipe_grid(nx, ny, 0.02, 0.02)
    dx, dy = spacing(g)
    i, j = np.arange(nx)[None, :], np.arange(ny)[:, None]
    Q = np.sin(np.pi * a * i / nx) * np.sin(np.pi * b * j / ny)
    n_total = 5.0
    lam = 4.0 * (np.sin(np.pi * a / (2 * nx)) ** 2 / dx ** 2 + np.sin(np.pi * b / (2 * ny)) ** 2 / dy ** 2)
    want = Q / (n_total * dx * dy) / lam
    u = orc.poisson(Q, g, n_total)
    assert np.abs(u - want).max() < 1e-13 * np.abs(want).max()


def test_dirichlet_point_charge_symmetry_and_sign(orc):
    """A positive charge mid-pipe: potential positive, maximal at the charge, symmetric about it, zero on the wall;
    and smaller everywhere than the open-boundary potential difference would allow (image charges pull it down)."""
    n = 32
    g = pipe_grid(n, n, 0.01, 0.01)
    Q = np.zeros((n, n))
    Q[16, 16] = 1.0                                            # node 16 = middle between the walls 0 and 32
    u = orc.poisson(Q, g, 1.0)
    assert u.max() == u[16, 16] > 0.0
    assert np.all(u[1:, 1:] > 0.0)
    assert np.abs(u[1:, 1:] - u[1:, 1:][::-1, :]).max() < 1e-14 * u.max()      # mirror about node 16
    assert np.abs(u[1:, 1:] - u[1:, 1:][:, ::-1]).max() < 1e-14 * u.max()
    assert np.abs(u[1:, 1:] - u[1:, 1:].T).max() < 1e-14 * u.max()
    assert np.abs(u[0, :]).max() < 1e-15 and np.abs(u[:, 0]).max() < 1e-15


def test_scnode_uses_the_pipe_solver_when_asked(orc):
    """track() through one SC node with boundary = 1: the work grids are those of the pipe solver."""
    from workloads import SCNODE, make_config
    wl = make_config(1, n=2000)
    wl.grids[0]["boundary"] = 1
    first = int(np.argmax(wl.kind == SCNODE)) + 1
    _, works = orc.track_workload(wl, stop_after_rows=first)
    w = works[0]
    u = orc.poisson(w.Q.reshape(64, 64), wl.grids[0], float(wl.n))
    assert np.array_equal(u.ravel(), w.u)
    g0 = dict(wl.grids[0], boundary=0)
    assert np.abs(orc.poisson(w.Q.reshape(64, 64), g0, float(wl.n)).ravel() - w.u).max() > 1e-3 * np.abs(w.u).max()
