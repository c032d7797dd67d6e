"""Helpers for the -m gpu parity tests: build the CUDA Grid and the oracle Problem from the same seeded inputs."""
import numpy as np

import fe_inputs as fi
from oracle import fe_oracle as orc


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    nb = np.linalg.norm(b.ravel())
    return np.linalg.norm((a - b).ravel()) / (nb if nb > 0 else 1.0)


def oracle_problem(w: fi.Workload, member: int = 0) -> orc.Problem:
    return orc.Problem(n=w.n, d=w.d, periodic=w.periodic, pbc_images=w.pbc_images, materials=w.materials[member],
                       g=w.globals_[member], matmap=w.matmap)


def workload_from_random(seed, n, periodic, pbc_images, dtype="f64", batch=1, **kw) -> fi.Workload:
    """fe_inputs.random_problem (heterogeneous, 3 materials incl. vacuum, Gm != 0, 8th-order slots, E_ext)
    wrapped as a Workload; batch members differ by seed."""
    qs = [fi.random_problem(seed + 7 * b, n=n, periodic=periodic, pbc_images=pbc_images, **kw) for b in range(batch)]
    q0 = qs[0]
    P = np.stack([q["P"] * (np.array([m.active for m in q0["materials"]])[q0["matmap"]])[None] for q in qs])
    return fi.Workload(name="random", n=n, d=q0["d"], periodic=periodic, pbc_images=pbc_images, batch=batch,
                       dtype=dtype, materials=[q["materials"] for q in qs], globals_=[q["globals_"] for q in qs],
                       matmap=q0["matmap"], P0=P, dt=1e-3, integrator=fi.EULER)
