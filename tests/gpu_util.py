"""Shared helpers for the -m gpu parity tests (marshalling between numpy canonical arrays and libdwf)."""
import numpy as np
import torch

import dwf_inputs as gen
from paper_2103_05034_b200 import Dwf, DWF_F32, DWF_F64

M5 = 1.8
TOL_APPLY = {"f64": 1e-12, "f32": 1e-5}       # BASELINE.json north_star: relative L2 per operator apply
TOL_CHEB = {"f64": 1e-11, "f32": 1e-4}        # order-64 Chebyshev: 1e-4 fp32 (north_star); fp64: 64 x apply


def rel_l2(got: np.ndarray, want: np.ndarray) -> float:
    """R18: max over rhs of ||got - want||_2 / ||want||_2."""
    worst = 0.0
    for r in range(want.shape[0]):
        worst = max(worst, np.linalg.norm((got[r] - want[r]).ravel()) / np.linalg.norm(want[r].ravel()))
    return worst


class Rig:
    """A handle plus the canonical inputs both sides see (rounded once to the run precision, R17)."""

    def __init__(self, L, Ls, prec, mass=0.01, seed_U=1000, unit_links=False, ws_nrhs=1):
        self.L, self.Ls, self.prec, self.mass = tuple(L), Ls, prec, mass
        U = gen.gauge_unit(L) if unit_links else gen.gauge_random(L, seed_U)
        self.U = gen.round_to_precision(U, prec)                       # complex128, what the oracle sees
        self.d = Dwf(L, Ls, M5, mass, DWF_F32 if prec == "f32" else DWF_F64)
        self.d.set_gauge(self.to_dev(self.U))
        self.d.set_workspace(ws_nrhs)

    def to_dev(self, a: np.ndarray) -> torch.Tensor:
        return torch.from_numpy(np.ascontiguousarray(a)).to(self.d.cdtype).cuda().contiguous()

    def spinor(self, nrhs, seed):
        return gen.round_to_precision(gen.spinor_gaussian(self.L, self.Ls, nrhs, seed), self.prec)

    def native(self, psi: np.ndarray, parity=-1) -> torch.Tensor:
        return self.d.import_(self.to_dev(psi), parity=parity)

    def canonical(self, native: torch.Tensor, nrhs, parity=-1) -> np.ndarray:
        return self.d.export(native, nrhs, parity=parity).cpu().numpy().astype(np.complex128)

    def apply(self, op, psi: np.ndarray, half=False) -> np.ndarray:
        nrhs = psi.shape[0]
        parity = 0 if half else -1
        x = self.native(psi, parity)
        y = self.d.field(nrhs, half=half)
        self.d.apply(op, x, y, nrhs)
        return self.canonical(y, nrhs, parity)
