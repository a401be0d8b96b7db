"""Adapters between a ``workloads.Workload`` and the two implementations under test."""
import numpy as np
import torch

import oracle


def np_(t):
    return None if t is None else t.detach().cpu().numpy()


def courant_xyz(w):
    """Courant components of the present dimensions mapped on (x, y, z)."""
    dims = [d for d, n in zip("xyz", (w.init["nx"], w.init["ny"], w.init["nz"])) if n > 0]
    out = dict(x=None, y=None, z=None)
    for d, c in zip(dims, w.courants):
        out[d] = c
    return out


def make_oracle(w, threads=1, **override):
    init = dict(w.init)
    init.update(override)
    o = oracle.Oracle(**init)
    o.set_threads(threads)
    c = courant_xyz(w)
    o.set_fields(th=np_(w.th).ravel(), rv=np_(w.rv).ravel(), rhod=np_(w.rhod).ravel(),
                 cx=None if c["x"] is None else np_(c["x"]).ravel(),
                 cy=None if c["y"] is None else np_(c["y"]).ravel(),
                 cz=None if c["z"] is None else np_(c["z"]).ravel())
    s = w.state
    o.set_state(np_(s["n"]).astype(np.uint64), np_(s["rw2"]), np_(s["rd3"]), np_(s["kappa"]),
                x=np_(s["x"]), y=np_(s["y"]), z=np_(s["z"]), id=np_(s["id"]).astype(np.uint32))
    return o


def make_particles(w, max_sd=None, **override):
    from paper_1310_1905_b200 import binding

    init = dict(w.init)
    init.update(override)
    p = binding.Particles(max_sd=max_sd or max(w.n_sd, 1), sd_conc_mean=w.meta.get("sd_per_cell", 0.0), **init)
    dev = "cuda"
    s = {k: (None if v is None else v.to(dev)) for k, v in w.state.items()}
    cs = [c.to(dev) for c in w.courants] + [None] * (3 - len(w.courants))
    p.init_from_arrays(w.rhod.to(dev), s["n"], s["rw2"], s["rd3"], s["kappa"], s["x"], s["y"], s["z"], s["id"],
                       courant_1=cs[0], courant_2=cs[1], courant_3=cs[2])
    return p, w.th.to(dev).clone(), w.rv.to(dev).clone()


def sorted_by_id(state):
    """dict of numpy arrays ordered by SD id (storage order is implementation-defined)."""
    st = {k: (v.detach().cpu().numpy() if isinstance(v, torch.Tensor) else np.asarray(v)) for k, v in state.items()}
    order = np.argsort(st["id"].astype(np.uint32), kind="stable")
    return {k: v[order] for k, v in st.items()}
