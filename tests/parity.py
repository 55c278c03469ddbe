"""Error norms of the parity protocol (reading R25 in DESIGN.md) and small helpers shared by the GPU tests."""
import numpy as np


def field_err(got, ref):
    """max |got - ref| / max |ref| per gas field; the three momentum components are normalised jointly."""
    got = np.asarray(got, dtype=np.float64); ref = np.asarray(ref, dtype=np.float64)
    e = {}
    e["rho"] = np.max(np.abs(got[0] - ref[0])) / np.max(np.abs(ref[0]))
    mscale = max(np.max(np.abs(ref[1:4])), 1e-300)
    e["mom"] = np.max(np.abs(got[1:4] - ref[1:4])) / mscale
    e["eps"] = np.max(np.abs(got[4] - ref[4])) / np.max(np.abs(ref[4]))
    return e


def part_err(got, ref, N):
    got = np.asarray(got, dtype=np.float64); ref = np.asarray(ref, dtype=np.float64)
    d = got[:3] - ref[:3]
    d -= N * np.round(d / N)
    e = {"x": np.max(np.abs(d)) / N if d.size else 0.0}
    e["w"] = (np.max(np.abs(got[3:] - ref[3:])) / max(np.max(np.abs(ref[3:])), 1e-300)) if d.size else 0.0
    return e


def rel_l2(got, ref):
    got = np.asarray(got, dtype=np.float64).ravel(); ref = np.asarray(ref, dtype=np.float64).ravel()
    return np.linalg.norm(got - ref) / max(np.linalg.norm(ref), 1e-300)


def rel_l2_trimmed(got, ref, frac=2e-4):
    """rel_l2 after dropping the `frac` largest-error entries.  The limiter gate (ab > 0), the energy floor and |v| make
    the step's derivative piecewise: a difference whose sign is decided at fp32 rounding level switches a few O(1)
    entries of the VJP (the fp64 oracle shows the same jumps when its input is perturbed by 1e-7).  Those entries are
    compared through the untrimmed north-star bound (<= 1e-3); everything else must agree tightly."""
    got = np.asarray(got, dtype=np.float64).ravel(); ref = np.asarray(ref, dtype=np.float64).ravel()
    err = np.abs(got - ref)
    k = int(np.ceil(frac * err.size))
    keep = np.argsort(err)[: err.size - k]
    return np.linalg.norm(err[keep]) / max(np.linalg.norm(ref), 1e-300)


def max_rel(got, ref):
    got = np.asarray(got, dtype=np.float64); ref = np.asarray(ref, dtype=np.float64)
    return np.max(np.abs(got - ref)) / max(np.max(np.abs(ref)), 1e-300)


def oracle_params(O, cfg, **kw):
    args = dict(n_part_side=cfg.n_side, H0=cfg.H0, Omega_m=cfg.Omega_m, Omega_b=cfg.Omega_b, Omega_L=cfg.Omega_L,
                static_mode=cfg.static_mode, gravity_on=cfg.gravity_on, e_floor=cfg.e_floor(), lim_eps=cfg.lim_eps)
    args.update(kw)
    return O.make_params(cfg.N, cfg.box, cfg.gamma, **args)


def shock_radii(rho):
    """Position of the density maximum of a centred blast wave (cell units): along the angle-averaged radial profile
    (0.5-cell bins) and along 9 rays (axes, face and body diagonals).  Returns (profile_peak, ray_min, ray_max)."""
    rho = np.asarray(rho, dtype=np.float64)
    N = rho.shape[0]
    c = N // 2
    q = np.arange(N) + 0.5 - (c + 0.5)
    z, y, x = np.meshgrid(q, q, q, indexing="ij")
    r = np.sqrt(x * x + y * y + z * z)
    bins = np.arange(0, N // 2, 0.5)
    idx = np.digitize(r.ravel(), bins)
    prof = np.bincount(idx, weights=rho.ravel(), minlength=len(bins) + 1) / np.maximum(np.bincount(idx, minlength=len(bins) + 1), 1)
    peak = bins[np.argmax(prof[1:])] + 0.25
    rays = []
    for dv in [(1, 0, 0), (0, 1, 0), (0, 0, 1), (1, 1, 0), (1, 0, 1), (0, 1, 1), (1, 1, 1), (-1, 1, 0), (1, -1, 1)]:
        dv = np.array(dv, float) / np.linalg.norm(dv)
        ss = np.arange(0, N / 2 - 2, 0.25)
        ii = np.floor((c + 0.5) + np.outer(ss, dv)).astype(int)
        rays.append(ss[np.argmax(rho[ii[:, 2], ii[:, 1], ii[:, 0]])])
    return peak, min(rays), max(rays)


def golden(name):
    """A text fixture under tests/golden/ (name value per line, '#' comments carry the citation) as a dict of floats."""
    import os
    out = {}
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", name)) as f:
        for line in f:
            line = line.strip()
            if line and not line.startswith("#"):
                k, v = line.split()[:2]
                out[k] = float(v)
    return out


# ---- conditioning of a piecewise-differentiable reference (reading R28) --------------------------------
def nonuniform_mask(gas, reach=4):
    """Cells that have a neighbour within `reach` cells along some axis (periodic) whose state differs in any field.
    Where the input is exactly constant over the stencil every flux difference is exactly 0 in any precision (identical
    inputs give identical outputs), so rounding cannot act there; everywhere else it can."""
    gas = np.asarray(gas)
    m = np.zeros(gas.shape[1:], dtype=bool)
    for ax in (1, 2, 3):
        for s in range(1, reach + 1):
            d = np.any(gas != np.roll(gas, s, axis=ax), axis=0)
            m |= d | np.roll(d, -s, axis=ax - 1)
    return m


def perturb_like_fp32(gas, seed, rel=6e-8):
    """The fp32 input promoted to fp64 and moved by one fp32 rounding (relative 6e-8, Gaussian) wherever rounding can
    act (nonuniform_mask): the model of what fp32 arithmetic does to the limiter / floor / |v| switches."""
    g = np.asarray(gas, dtype=np.float64)
    rng = np.random.default_rng(seed)
    return g * (1.0 + rel * rng.standard_normal(g.shape) * nonuniform_mask(gas)[None])


def stable_entries(ref, perturbed_refs, tol=1e-5):
    """Entries of a reference gradient that the reference itself reproduces to tol x max|ref| when its input moves by one
    fp32 rounding.  On these a correct fp32 adjoint must agree tightly; the others sit on a switch of the piecewise
    derivative, where the one-sided values differ by O(1) and any of them is valid."""
    ref = np.asarray(ref, dtype=np.float64)
    scale = np.max(np.abs(ref))
    ok = np.ones(ref.shape, dtype=bool)
    for r in perturbed_refs:
        ok &= np.abs(np.asarray(r, dtype=np.float64) - ref) <= tol * scale
    return ok


def masked_errors(got, ref, mask):
    """(max |got - ref| / max |ref|, relative L2) over the entries selected by mask."""
    got = np.asarray(got, dtype=np.float64); ref = np.asarray(ref, dtype=np.float64)
    d = (got - ref)[mask]
    return np.max(np.abs(d)) / np.max(np.abs(ref)), np.linalg.norm(d) / max(np.linalg.norm(ref[mask]), 1e-300)
