"""ORACLE (test infrastructure, like the rest of this package): ePIE-minibatch and the LSQML-style joint step with SUB-PIXEL scan positions.

SURVEY.md 8(f) f4 / R10 ("sub-pixel shifts = NEXT f4").  PAPER.md does not say how ptychopy treats the fractional
part of a position; reading R28 of DESIGN.md fixes it as the textbook rule -- the Fourier shift theorem applied to
the PROBE -- and this file is that rule written out in fp64 numpy, step by step.  Frame j sits at r_j + delta_j,
r_j the integer corner (as everywhere else), delta_j = (dy, dx) in [0, 1)^2:

    S_d[f]   = F^-1[ F[f](k) exp(-2 pi i (k_y d_y + k_x d_x) / N) ],  k = numpy.fft.fftfreq(N) N  (signed; Nyquist = -N/2)
    P_jk     = S_{delta_j}[P_k]                      the probe as frame j sees it (periodic Fourier interpolation)
    psi_jk   = P_jk O_j,  Phi = F psi,  Phi' = Pi_M Phi (R2, R3, R6: oracle.modulus_project, the C oracle's routine),
    chi_jk   = F^-1 Phi' - psi_jk
    n_O(r_j + r) += sum_k conj(P_jk) chi_jk          d_O(r_j + r) += sum_k |P_jk|^2
    n_Pk         += S_{-delta_j}[ conj(O_j) chi_jk ]  (the adjoint of the shift brings the term back into the probe's frame)
    d_P          += |O_j|^2                           (not shifted: a positive normaliser; Fourier interpolation could make it negative)
    dO = n_O / (d_O + delta_O max_r sum_k |P_k|^2)    (R8; the regulariser from the UNSHIFTED probe)
    dP_k = n_Pk / (d_P + delta_P max_r d_P),   O += alpha_O dO,   P_k += alpha_P dP_k (if the probe is updated)

With every delta_j = 0 this is orc_minibatch_step(EPIE_MB) of ptycho_oracle.c (pinned so in tests/test_oracle_pins.py, together
with the shift against its closed form on a Fourier mode, S_d S_{1-d} = a roll by one pixel, the common-shift equivalence with a
pre-shifted probe, and the back-shift of the probe term).  Library primitives used as steps: numpy.fft, oracle.modulus_project.
"""
from __future__ import annotations

import numpy as np

from . import DEFAULTS, batches, modulus_project, to_real_intensity


def shift(f: np.ndarray, dy: float, dx: float) -> np.ndarray:
    """S_(dy,dx)[f] on the last two axes: f moved by +dy rows and +dx columns (periodic Fourier interpolation)."""
    n = f.shape[-1]
    k = np.fft.fftfreq(n) * n
    ramp = np.exp(-2j * np.pi * (k[:, None] * dy + k[None, :] * dx) / n)
    return np.fft.ifft2(np.fft.fft2(np.asarray(f, np.complex128)) * ramp)


def epie_mb_step(O, P, pos, frac, inten, frames, update_probe, par, lsqml=False, steps_out=None):
    """One minibatch step over `frames` (in place on O, P; fp64).  Returns the batch's error term sum (sqrt I - A)^2.
    lsqml = True: the joint step (a, b) of R9 instead of the fixed (alpha_O, alpha_P), its five sums taken from their per-frame
    DEFINITIONS with the shifted probes and the shifted probe direction:
        u_jk = P_jk dO_j,   v_jk = S_{delta_j}[dP_k] O_j   (O_j the object BEFORE the step),   c = chi_jk
        A11 = sum |u|^2, A22 = sum |v|^2, A12 = Re sum conj(u) v, b1 = Re sum conj(u) c, b2 = Re sum conj(v) c
        l = 1 + lambda;  probe updated: (a, b) solve [[A11 l, A12], [A12, A22 l]] (a, b)^T = (b1, b2)^T (0, 0 if singular);
        otherwise a = b1 / (A11 l), b = 0      -- exactly the rule of orc_minibatch_step."""
    K, n = P.shape[0], P.shape[-1]
    nO = np.zeros_like(O)
    dO = np.zeros(O.shape)
    nP = np.zeros_like(P)
    dP = np.zeros((n, n))
    err = 0.0
    kept = []
    for j in frames:
        y, x = int(pos[j, 0]), int(pos[j, 1])
        dy, dx = float(frac[j, 0]), float(frac[j, 1])
        Oj = O[y:y + n, x:x + n]
        Pj = shift(P, dy, dx)                                            # (K, n, n)
        psi = Pj * Oj[None]
        Phi = np.fft.fft2(psi)
        Phi2, e = modulus_project(Phi, inten[j], par["pbound"])
        err += e
        chi = np.fft.ifft2(Phi2) - psi
        if lsqml:
            kept.append((Pj, chi, Oj.copy()))
        nO[y:y + n, x:x + n] += np.sum(np.conj(Pj) * chi, axis=0)
        dO[y:y + n, x:x + n] += np.sum(np.abs(Pj) ** 2, axis=0)
        nP += shift(np.conj(Oj)[None] * chi, -dy, -dx)
        dP += np.abs(Oj) ** 2
    maxP = float(np.max(np.sum(np.abs(P) ** 2, axis=0)))
    dirO = nO / (dO + par["delta_obj"] * maxP)
    dirP = nP / (dP + par["delta_probe"] * float(np.max(dP)))[None]
    sa, sb = par["alpha_obj"], (par["alpha_probe"] if update_probe else 0.0)
    if lsqml:
        A11 = A22 = A12 = b1 = b2 = 0.0
        for j, (Pj, chi, Oj) in zip(frames, kept):
            y, x = int(pos[j, 0]), int(pos[j, 1])
            u = Pj * dirO[None, y:y + n, x:x + n]
            v = shift(dirP, float(frac[j, 0]), float(frac[j, 1])) * Oj[None]
            A11 += float(np.sum(np.abs(u) ** 2)); A22 += float(np.sum(np.abs(v) ** 2))
            A12 += float(np.sum((np.conj(u) * v).real))
            b1 += float(np.sum((np.conj(u) * chi).real)); b2 += float(np.sum((np.conj(v) * chi).real))
        l = 1.0 + par["lsq_lambda"]
        if not update_probe:
            sa, sb = (b1 / (A11 * l) if A11 > 0 else 0.0), 0.0
        else:
            det = A11 * l * A22 * l - A12 * A12
            if not (det > 0) or not np.isfinite(det):
                sa, sb = 0.0, 0.0
            else:
                sa, sb = (b1 * A22 * l - A12 * b2) / det, (A11 * l * b2 - A12 * b1) / det
    O += sa * dirO
    if update_probe:
        P += sb * dirP
    if steps_out is not None:
        steps_out.append((sa, sb))
    return err


def dm_iteration(O, P, psi, pos, frac, inten, eps_O, eps_P, update_probe, pbound):
    """One DM iteration with sub-pixel positions, in place on O, P, psi (J, K, n, n); the steps of orc_dm_iteration (SURVEY 8(c)
    "DM" 1-5; R4 lagged probe sums, R5 blends, R6) with P_jk = S_{delta_j}[P_k] in place of P_k and the probe term shifted back:
        1  n_Pk += S_{-delta_j}[conj(O_j) psi_jk],  d_P += |O_j|^2                 (incoming psi, current O)
        2  psi_O = P_jk O_j;  Phi = F[2 psi_O - psi_j];  Phi' = Pi_M Phi;  psi_F = F^-1 Phi'
        3  psi_j <- psi_j + psi_F - psi_O
        4  n_O += sum_k conj(P_jk) psi_jk,  d_O += sum_k |P_jk|^2                  (new psi, current P)
        5  O <- (n_O + eps_O O)/(d_O + eps_O);  P_k <- (n_Pk + eps_P P_k)/(d_P + eps_P) if the probe is updated
    Returns the error term sum.  (d_P is not shifted, as in the minibatch step: a shift does not commute with the multiplication
    by |O_j|^2, so with the probe updated the ground truth is a fixed point only up to the variation of |O_j|^2 over a pixel;
    with the probe frozen it is one exactly -- pinned.)"""
    K, n = P.shape[0], P.shape[-1]
    nP = np.zeros_like(P); dP = np.zeros((n, n)); nO = np.zeros_like(O); dO = np.zeros(O.shape)
    for j, (y, x) in enumerate(pos):
        Oj = O[y:y + n, x:x + n]
        nP += shift(np.conj(Oj)[None] * psi[j], -float(frac[j, 0]), -float(frac[j, 1]))
        dP += np.abs(Oj) ** 2
    err = 0.0
    for j, (y, x) in enumerate(pos):
        Pj = shift(P, float(frac[j, 0]), float(frac[j, 1]))
        psiO = Pj * O[None, y:y + n, x:x + n]
        Phi2, e = modulus_project(np.fft.fft2(2 * psiO - psi[j]), inten[j], pbound)
        err += e
        psi[j] = psi[j] + np.fft.ifft2(Phi2) - psiO
        nO[y:y + n, x:x + n] += np.sum(np.conj(Pj) * psi[j], axis=0)
        dO[y:y + n, x:x + n] += np.sum(np.abs(Pj) ** 2, axis=0)
    O[...] = (nO + eps_O * O) / (dO + eps_O)
    if update_probe:
        P[...] = (nP + eps_P * P) / (dP + eps_P)[None]
    return err


class SubpixelOracle:
    """State and sequencing (batches R8, probe_start, error history C3), mirroring oracle.Oracle for EPIE_MB."""

    def __init__(self, obj, probe, pos, frac, intensities, params=None):
        self.par = dict(DEFAULTS)
        self.par.update(params or {})
        self.O = np.array(obj, np.complex128)
        self.P = np.array(probe, np.complex128)
        if self.P.ndim == 2:
            self.P = self.P[None]
        self.pos = np.asarray(pos, np.int64).reshape(-1, 2)
        self.frac = np.asarray(frac, np.float64).reshape(-1, 2)
        assert self.frac.shape == self.pos.shape and (self.frac >= 0).all() and (self.frac < 1).all()
        self.inten = intensities                                        # uint16 / float32 as given (masks: R3)
        it = to_real_intensity(intensities, np.float64)
        self.sum_I = float(np.sum(it[it >= 0]))
        self.t = 0
        self.err: list[float] = []
        self.steps: list[tuple[float, float]] = []
        self.psi = None
        d = self.par["delta_blend"]                                      # R5: fixed at init, from the unshifted probe
        self.eps_O = d * float(np.max(np.sum(np.abs(self.P) ** 2, axis=0)))
        self.eps_P = d * len(self.pos) * float(np.max(np.abs(self.O) ** 2))

    def eval_error(self) -> float:
        """C3 with the shifted probes: sum_j sum_q (sqrt I_j - A_j)^2 / sum I over unmasked pixels, A_j^2 = sum_k |F[P_jk O_j]|^2."""
        n = self.P.shape[-1]
        num = 0.0
        for j, (y, x) in enumerate(self.pos):
            Phi = np.fft.fft2(shift(self.P, *self.frac[j]) * self.O[None, y:y + n, x:x + n])
            num += modulus_project(Phi, self.inten[j], 0.0)[1]
        return num / (self.sum_I if self.sum_I > 0 else 1.0)

    def iterate(self, n_iters: int = 1, alg: str = "EPIE_MB"):
        assert alg in ("EPIE_MB", "LSQML", "DM")
        p = self.par
        n = self.P.shape[-1]
        for _ in range(n_iters):
            upd = self.t >= p["probe_start"]
            num = 0.0
            if alg == "DM":
                if self.psi is None:                                     # R4: psi_j = P_jk O_j before the first DM iteration
                    self.psi = np.stack([shift(self.P, *self.frac[j]) * self.O[None, y:y + n, x:x + n] for j, (y, x) in enumerate(self.pos)])
                num = dm_iteration(self.O, self.P, self.psi, self.pos, self.frac, self.inten, self.eps_O, self.eps_P, upd, p["pbound"])
                self.err.append(num / (self.sum_I if self.sum_I > 0 else 1.0))
                self.t += 1
                continue
            self.psi = None
            for fr in batches(len(self.pos), p["batch_size"], p["batch_order"]):
                num += epie_mb_step(self.O, self.P, self.pos, self.frac, self.inten, fr, upd, p, lsqml=alg == "LSQML", steps_out=self.steps)
            self.err.append(num / (self.sum_I if self.sum_I > 0 else 1.0))
            self.t += 1
        return self
