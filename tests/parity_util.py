"""Helpers shared by the GPU parity tests: the error metric of DESIGN.md R17 and an oracle runner."""
import numpy as np

# north_star tolerances: (one step, 100 steps, dt)
TOL = {np.dtype(np.float64): (1e-12, 1e-9, 1e-13), np.dtype(np.float32): (1e-5, 1e-3, 1e-6)}


def field_errors(got, ref):
    """err_f = max_i |got_f - ref_f| / max_i |ref_f| per conserved field (R17).  Every field is
    measured on its OWN scale; only a momentum component that is identically ~0 in the reference (below 1e-12 of the
    largest component: a 1-D flow embedded in 2-D / 3-D, v = 0 initial data) borrows the scale max_b max_i |m_b|,
    because it has none of its own."""
    nf = ref.shape[0]
    g = got.reshape(nf, -1).astype(np.float64)
    r = ref.reshape(nf, -1).astype(np.float64)
    scale = np.abs(r).max(axis=1)
    mom = scale[1:nf - 1].max()
    scale[1:nf - 1] = np.where(scale[1:nf - 1] <= 1e-12 * mom, mom, scale[1:nf - 1])
    scale = np.where(scale > 0, scale, 1.0)
    return np.abs(g - r).max(axis=1) / scale


def own_scale_errors(got, ref):
    """SURVEY A17 read strictly: err_f = max_i |got_f - ref_f| / max_i |ref_f| with EACH field on its own scale, the
    momentum components too (config 1's m_y, max ~ 0.02 beside m_x ~ 1, is the tight case).  A field that is zero
    everywhere in the reference must be zero in `got` (error 0) or the error is infinite."""
    nf = ref.shape[0]
    g = got.reshape(nf, -1).astype(np.float64)
    r = ref.reshape(nf, -1).astype(np.float64)
    scale = np.abs(r).max(axis=1)
    diff = np.abs(g - r).max(axis=1)
    with np.errstate(divide="ignore", invalid="ignore"):
        return np.where(scale > 0, diff / np.where(scale > 0, scale, 1.0), np.where(diff > 0, np.inf, 0.0))


def oracle_steps(oracle_mod, w, nsteps, riemann="hllc", threads="omp", boundary=None, cfl=None):
    """Run the oracle nsteps steps with its own CFL dt; returns (state, [dt_k])."""
    o = oracle_mod.Oracle(w.n, w.extent, w.gamma, w.dtype, boundary or w.boundary, riemann, threads)
    o.set_state(w.U)
    dts = []
    for _ in range(nsteps):
        dts.append(o.cfl_dt(cfl or w.cfl))
        o.step(dts[-1])
    out = o.get_state()
    o.close()
    return out, dts
