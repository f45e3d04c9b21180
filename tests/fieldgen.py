"""Seeded synthetic input fields for the tests (shared by the oracle tests and the GPU parity tests).

Holds none of the method's arithmetic: no Laplacian, no potential, no update, no link counting --
only shapes, random numbers and analytic profiles used as *inputs*.  Arrays are indexed [z, y, x]
(3D) or [y, x] (2D), C-contiguous, so that the linear index is s = x + N*(y + N*z), x fastest.
"""
import numpy as np


def random_state(dims, N, seed, dtype=np.float32, amp=1.0, with_velocity=True):
    """phi uniform in (-amp, amp), phidot uniform in (-amp/2, amp/2); values are float32-exact so
    the float and double runs start from identical numbers (PAPER.md:113 protocol)."""
    rng = np.random.default_rng(seed)
    shape = (N,) * dims
    phi = rng.uniform(-amp, amp, shape).astype(np.float32).astype(dtype)
    if with_velocity:
        pd = rng.uniform(-0.5 * amp, 0.5 * amp, shape).astype(np.float32).astype(dtype)
    else:
        pd = np.zeros(shape, dtype)
    return phi, pd


def plane_wave(dims, N, modes, phase=0.0, amp=1.0, offset=0.0, dtype=np.float64):
    """offset + amp*cos(k.x + phase) with k_i = 2*pi*modes[i]/N; modes is given in (x, y[, z]) order."""
    ax = [np.arange(N, dtype=np.float64)] * dims
    grids = np.meshgrid(*ax, indexing="ij")          # grids[0] varies along axis 0 (= z or y)
    arg = np.zeros((N,) * dims)
    for i, m in enumerate(modes):                    # modes[0] -> x = last axis
        arg += (2.0 * np.pi * m / N) * grids[dims - 1 - i]
    return (offset + amp * np.cos(arg + phase)).astype(dtype)


def kink_pair(dims, N, kappa, phi0=1.0, dtype=np.float64, gamma=1.0, shift=0.0):
    """Planar wall + anti-wall normal to x at x1 = N/4 - 1/2 and x2 = 3N/4 - 1/2 (between sites):
    phi0*(tanh(g*k*(x-x1-shift)) - tanh(g*k*(x-x2+shift)) - 1), uniform in y (and z)."""
    x = np.arange(N, dtype=np.float64)
    x1, x2 = N / 4 - 0.5, 3 * N / 4 - 0.5
    prof = phi0 * (np.tanh(gamma * kappa * (x - x1 - shift)) - np.tanh(gamma * kappa * (x - x2 + shift)) - 1.0)
    return np.ascontiguousarray(np.broadcast_to(prof, (N,) * dims)).astype(dtype)


def roll_state(a, shifts):
    """Periodic translation by shifts given in (x, y[, z]) order."""
    dims = a.ndim
    out = a
    for i, sh in enumerate(shifts):
        out = np.roll(out, sh, axis=dims - 1 - i)
    return np.ascontiguousarray(out)


def flip_axis(a, axis_xyz):
    """Reflection x -> -x (site 0 fixed) along the axis given as 0=x, 1=y, 2=z."""
    ax = a.ndim - 1 - axis_xyz
    return np.ascontiguousarray(np.roll(np.flip(a, axis=ax), 1, axis=ax))
