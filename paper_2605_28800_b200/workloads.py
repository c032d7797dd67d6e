"""Drivers of the two BASELINE.json workloads that are schedules of fe_step calls rather than a single run:
the BaTiO3 temperature sweep (config 3, reading A12) and the bilayer field sweep (config 4, A13).
Every step of the path runs in the CUDA library; this module only sequences the calls (coefficient / field changes
between legs) and reads the observables the configs name from fe_energy (means) and a histogram of the state."""
from __future__ import annotations

from typing import Callable, Dict, List, Sequence

import numpy as np
import torch

from .binding import FE_EULER, FE_TERM_ALL, Grid


def phase_histogram(P: torch.Tensor, floor: float = 0.02) -> np.ndarray:
    """Per batch member: number of cells whose polarisation has 0 (|P| < floor: cubic), 1 (T), 2 (O) or 3 (R)
    components larger than 0.3 |P| (reading A12).  P: [B][3][nz][ny][nx] on the device, in the units of the run."""
    norm = torch.linalg.vector_norm(P, dim=1)
    ncomp = (P.abs() > 0.3 * norm.unsqueeze(1)).sum(dim=1)
    ncomp = torch.where(norm < floor, torch.zeros_like(ncomp), ncomp)
    B = P.shape[0]
    out = torch.stack([(ncomp.reshape(B, -1) == k).sum(dim=1) for k in range(4)], dim=1)
    return out.cpu().numpy()


def temperature_sweep(g: Grid, P: torch.Tensor, material_at: Callable[[int, int], object], n_legs: int,
                      steps_per_leg: int, dt: float, floor: float = 0.02) -> List[Dict[str, np.ndarray]]:
    """Config 3: leg l runs steps_per_leg Euler steps with member b at the material material_at(b, l); the state
    carries over, the tensor is not recomputed.  Returns per leg the mean |P| and the phase histogram per member."""
    log = []
    for leg in range(n_legs):
        for b in range(g.batch):
            g.set_material(b, 0, material_at(b, leg))
        g.step(P, dt, steps_per_leg, FE_EULER, FE_TERM_ALL)
        log.append({"mean_abs_P": torch.linalg.vector_norm(P, dim=1).mean(dim=(1, 2, 3)).cpu().numpy(),
                    "phases": phase_histogram(P, floor)})
    return log


def field_sweep(g: Grid, P: torch.Tensor, fields_z: Sequence[float], steps_per_point: int, dt: float,
                member: int = -1) -> np.ndarray:
    """Config 4: for every field point set E_ext = (0, 0, E_z), run steps_per_point Euler steps, record <Pz> over the
    active cells.  Returns [len(fields_z)][B] (the hysteresis loop <Pz>(E_z))."""
    loop = np.zeros((len(fields_z), g.batch))
    for k, ez in enumerate(fields_z):
        g.set_external_field(member, (0.0, 0.0, float(ez)))
        g.step(P, dt, steps_per_point, FE_EULER, FE_TERM_ALL)
        loop[k] = g.energy(P)[:, 7]
    return loop


def strain_sweep(g: Grid, P: torch.Tensor, materials: Sequence[object], steps_per_leg: int, dt: float,
                 material_id: int = 0) -> np.ndarray:
    """Strain study: leg l sets material `material_id` of every member to materials[l] (alpha_1z
    scaled by r_s) and relaxes for steps_per_leg Euler steps from the previous leg's state (adiabatic continuation).
    Returns per leg and member [<Px>, <Py>, <Pz>, <|Pz|> / <|P|>] over the cells of the whole grid."""
    out = np.zeros((len(materials), g.batch, 4))
    for leg, m in enumerate(materials):
        g.set_material(-1, material_id, m)
        g.step(P, dt, steps_per_leg, FE_EULER, FE_TERM_ALL)
        out[leg, :, :3] = g.energy(P)[:, 5:8]
        norm = torch.linalg.vector_norm(P, dim=1).mean(dim=(1, 2, 3))
        out[leg, :, 3] = (P[:, 2].abs().mean(dim=(1, 2, 3)) / norm.clamp_min(1e-300)).cpu().numpy()
    return out
