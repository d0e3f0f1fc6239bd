"""Shared helpers of the `-m gpu` parity tests: drive the CUDA path through the C ABI (python binding
of include/hr.h) and the oracle on the same seeded inputs.  No arithmetic of the method lives here."""
import numpy as np

import lattice_inputs as li
import oracle

BC_T = (-1, 1, 1, 1)             # periodic in space, antiperiodic in time (BASELINE.json:configs)
TOL = {"f64": 1e-13, "f32": 2e-6}  # BASELINE.json:north_star: relative L2 vs the fp64 oracle

# (N, rep name, oracle rep id)
COMBOS = [(2, "fund"), (2, "adj"), (2, "sym"), (3, "fund"), (3, "adj"), (3, "sym"), (3, "asym"), (4, "fund"), (4, "asym"), (4, "sym"), (4, "adj")]


def rel_l2(a, b):
    a = np.asarray(a).reshape(-1)
    b = np.asarray(b).reshape(-1)
    num = np.sqrt(np.sum(np.abs(a.astype(np.complex128) - b.astype(np.complex128)) ** 2))
    den = np.sqrt(np.sum(np.abs(b.astype(np.complex128)) ** 2))
    return float(num / den)


def oracle_rep_id(rep):
    return oracle.REP_NAMES[rep]


class GpuProblem:
    """One lattice + gauge field on the GPU (fundamental imported, represented via hr_represent_links)."""

    def __init__(self, hr, dims, N, rep, prec, U_fund, bc=BC_T, fund_prec=None):
        self.hr = hr
        self.prec = hr.PREC_NAMES[prec] if isinstance(prec, str) else prec
        self.lat = hr.Lattice(dims, bc, N, rep)
        fp = self.prec if fund_prec is None else (hr.PREC_NAMES[fund_prec] if isinstance(fund_prec, str) else fund_prec)
        self.fund = self.lat.gauge(False, fp)
        self.lat.import_gauge(self.fund, U_fund)
        self.links = self.lat.gauge(True, self.prec)
        self.lat.represent_links(self.links, self.fund)

    def represented(self):
        return self.lat.export_gauge(self.links, True, self.hr.HR_F64)

    def dphi_eo(self, psi_half, parity):
        inp = self.lat.spinor(self.prec)
        out = self.lat.spinor(self.prec)
        out.fill_(0xFF)  # NaN pattern: every byte of the output must be written by the kernel
        self.lat.import_spinor(inp, self.prec, psi_half, 1 - parity)
        self.lat.dphi_eo(out, inp, self.links, parity)
        return self.lat.export_spinor(out, self.prec, parity)

    def dirac(self, m0, psi_eo):
        vh = self.lat.vh
        half = self.hr.hr_spinor_bytes(self.lat.ctx, self.prec)
        inp = self.lat.spinor(self.prec, full=True)
        out = self.lat.spinor(self.prec, full=True)
        out.fill_(0xFF)
        for p in (0, 1):
            self.lat.import_spinor(inp[p * half:(p + 1) * half], self.prec, psi_eo[p * vh:(p + 1) * vh], p)
        self.lat.dirac(m0, out, inp, self.links)
        return np.concatenate([self.lat.export_spinor(out[p * half:(p + 1) * half], self.prec, p) for p in (0, 1)], axis=0)

    def close(self):
        self.lat.close()


def make_inputs(dims, N, seed_links, seed_spinor, d, kind="haar"):
    U = li.haar_links(seed_links, N, dims) if kind == "haar" else li.near_identity_links(seed_links, N, dims, 0.3)
    psi = li.gaussian_spinor(seed_spinor, li.volume(dims) // 2, d)
    return U, psi
