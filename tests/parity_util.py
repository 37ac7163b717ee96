"""Shared helpers of the GPU-vs-oracle parity tests (test infrastructure)."""
import numpy as np


def rel_err(gpu, ref):
    """Per-field norm of SURVEY 8(c): max|gpu - ref| / max|ref| (vectors as one field)."""
    gpu = np.asarray(gpu, dtype=np.float64)
    den = np.abs(ref).max()
    num = np.abs(gpu - ref).max()
    if den == 0.0:
        return num
    return num / den


def run_oracle(ref, cfg, steps_list):
    """Oracle outputs (rho, p, u, phi, state) after each cumulative step count in steps_list."""
    nz, ny, nx = cfg["shape"]
    sim = ref.RefSim(nx, ny, nz, ref.make_params(**cfg["params"]))
    sim.init(cfg["phi"], cfg["u"])
    out, done = [], 0
    for s in steps_list:
        sim.step(s - done)
        done = s
        out.append(dict(zip(("rho", "p", "u", "phi"), sim.get())) | {"state": sim.get_state()})
    sim.close()
    return out


def run_gpu(cfg, steps_list, precision="f64", flags=0, host_api=False):
    from paper_2501_00846_b200 import binding as B
    nz, ny, nx = cfg["shape"]
    s = B.Solver(nx, ny, nz, cfg["params"], precision=precision, flags=flags)
    npdt = np.float64 if precision == "f64" else np.float32
    if host_api:
        s.init_host(np.ascontiguousarray(cfg["phi"], dtype=npdt),
                    np.ascontiguousarray(cfg["u"], dtype=npdt))
    else:
        s.init(cfg["phi"], cfg["u"])
    out, done = [], 0
    for n in steps_list:
        s.step(n - done)
        done = n
        if host_api:
            h = dict(rho=np.empty(s.shape, npdt), p=np.empty(s.shape, npdt),
                     u=np.empty((3,) + s.shape, npdt), phi=np.empty(s.shape, npdt))
            s.get_host(h)
            out.append(h)
        else:
            g = s.get()
            st = s.get_state()
            s.synchronize()
            d = {k: v.cpu().numpy() for k, v in g.items()}
            d["state"] = {k: v.cpu().numpy() for k, v in st.items()}
            out.append(d)
    launches = s.launches
    s.close()
    return out, launches


def ahat_ref(ref, cfg, state):
    """(1 - omega(phi)) a2_neq of the oracle state: what the CUDA path stores."""
    ps, u, A, a, phi = state
    prm = ref.make_params(**cfg["params"])
    om = np.vectorize(lambda x: ref.omega(prm, x))(phi)
    return (1.0 - om)[None] * A


def compare(ref, cfg, g, r, tol, fields=("rho", "p", "u", "phi"), state_tol=None):
    errs = {k: rel_err(g[k], r[k]) for k in fields}
    if state_tol is not None and "state" in g:
        ps, u, A, a, phi = r["state"]
        errs["pstar"] = rel_err(g["state"]["pstar"], ps)
        errs["a"] = rel_err(g["state"]["a"], a)
        errs["Ahat"] = rel_err(g["state"]["A"], ahat_ref(ref, cfg, r["state"]))
    bad = {k: v for k, v in errs.items()
           if not (v <= (state_tol if k in ("pstar", "a", "Ahat") else tol))}
    return errs, bad
