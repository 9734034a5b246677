"""Seeded synthetic Hamiltonians shaped like BASELINE.json's five configs.

This module holds NONE of the method's arithmetic (no SP2, no bounds, no
density matrix): it only draws inputs.  It is the one module that serves both
the CUDA path's tests/bench and the CPU oracle's tests; it imports neither.

The paper's inputs are LATTE SCC-DFTB Hamiltonians of periodic water boxes
(PAPER.md:178); neither LATTE nor those matrices exist here, so these matrices
take their shapes (N = 6 orbitals x molecules, 4 occupied per molecule, dense
symmetric, gapped spectrum) and stand in for them.

Recipe (all float64, ``rng = np.random.default_rng(seed)``, draws in this order):
    G      <- rng.standard_normal((N, N))
    Q, R   <- qr(G);  Q <- Q * sign(diag R)           (Haar-distributed orthogonal Q)
    lam_o  <- rng.uniform(occ_lo, occ_hi, n_occ)       occupied eigenvalues
    lam_u  <- rng.uniform(un_lo,  un_hi,  N - n_occ)   unoccupied eigenvalues
    H      <- (Q * lam) Q^T;  H <- (H + H^T)/2
    H1     <- 1e-2 * (G1 + G1^T)/sqrt(2),  G1 <- rng.standard_normal((N, N))   (response configs)
    P      <- (G2 + G2^T)/sqrt(2N),        G2 <- rng.standard_normal((N, N))   (MD-sequence config)
seed = 20210714 + config index.  ``in_dtype`` float32 configs round H (and H1, P)
to fp32 ONCE here, so the oracle and the GPU solve the same rounded problem.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

BASE_SEED = 20210714


@dataclass(frozen=True)
class Sp2Config:
    name: str
    index: int
    n: int
    n_occ: int
    occ: tuple          # (lo, hi) of occupied eigenvalues
    unocc: tuple        # (lo, hi) of unoccupied eigenvalues
    in_dtype: str       # "f64" | "f32"
    response: bool
    n_steps: int = 1    # MD-sequence length (config 5)

    @property
    def seed(self):
        return BASE_SEED + self.index

    @property
    def gap(self):
        return self.unocc[0] - self.occ[1]


CONFIGS = {
    1: Sp2Config("tiny_n128", 1, 128, 64, (-2.0, -0.5), (0.5, 2.0), "f64", False),
    2: Sp2Config("n1024_response", 2, 1024, 512, (-1.5, -0.25), (0.25, 1.5), "f64", True),
    3: Sp2Config("waterbox_n6000_f32", 3, 6000, 4000, (-1.2, -0.1), (0.1, 1.2), "f32", False),
    4: Sp2Config("smallgap_n8192", 4, 8192, 4096, (-1.0, -0.025), (0.025, 1.0), "f64", True),
    5: Sp2Config("md_sequence_n16384", 5, 16384, 8192, (-1.0, -0.1), (0.1, 1.0), "f32", False, 50),
}


def scaled_config(cfg: Sp2Config, n: int, name: str | None = None) -> Sp2Config:
    """Same spectrum/occupation fraction at a different N (parity-test sizes)."""
    n_occ = (cfg.n_occ * n) // cfg.n
    return Sp2Config(name or f"{cfg.name}_at_{n}", cfg.index, n, n_occ, cfg.occ, cfg.unocc,
                     cfg.in_dtype, cfg.response, cfg.n_steps)


def _np_dtype(in_dtype):
    return np.float32 if in_dtype == "f32" else np.float64


def _haar_q_numpy(G):
    Q, R = np.linalg.qr(G)
    s = np.sign(np.diag(R))
    s[s == 0] = 1.0
    return Q * s[None, :]


def _haar_q_and_h_torch(G, lam, device):
    """Same algebra as the NumPy path, on a CUDA device in float64 (input
    generation only -- bench/tests may use torch; the library may not)."""
    import torch

    Gd = torch.from_numpy(G).to(device)
    Q, R = torch.linalg.qr(Gd)
    del Gd
    s = torch.sign(torch.diagonal(R))
    s[s == 0] = 1.0
    del R
    Q = Q * s[None, :]
    lamd = torch.from_numpy(lam).to(device)
    H = (Q * lamd[None, :]) @ Q.T
    H = 0.5 * (H + H.T)
    return Q.cpu().numpy(), H.cpu().numpy()


def make_problem(cfg: Sp2Config, seed: int | None = None, device: str = "cpu",
                 want_h1: bool | None = None, want_p: bool = False):
    """Draw one problem.  Returns a dict:
        H (n x n, cfg dtype), Q (f64), lam (f64, lam[k] belongs to column k of Q),
        n, n_occ, and optionally H1 / P (cfg dtype).
    ``device="cuda"`` only moves the QR and the two GEMMs of the recipe to the
    GPU (float64, torch); the random draws are identical.
    """
    rng = np.random.default_rng(cfg.seed if seed is None else seed)
    n, n_occ = cfg.n, cfg.n_occ
    G = rng.standard_normal((n, n))
    lam_o = rng.uniform(cfg.occ[0], cfg.occ[1], n_occ)
    lam_u = rng.uniform(cfg.unocc[0], cfg.unocc[1], n - n_occ)
    lam = np.concatenate([lam_o, lam_u])
    if device == "cpu":
        Q = _haar_q_numpy(G)
        del G
        H = (Q * lam[None, :]) @ Q.T
        H = 0.5 * (H + H.T)
    else:
        Q, H = _haar_q_and_h_torch(G, lam, device)
        del G
    dt = _np_dtype(cfg.in_dtype)
    out = dict(H=np.ascontiguousarray(H.astype(dt)), Q=Q, lam=lam, n=n, n_occ=n_occ, cfg=cfg)
    if cfg.response if want_h1 is None else want_h1:
        G1 = rng.standard_normal((n, n))
        out["H1"] = np.ascontiguousarray((1e-2 * (G1 + G1.T) / math.sqrt(2.0)).astype(dt))
        del G1
    if want_p:
        G2 = rng.standard_normal((n, n))
        out["P"] = np.ascontiguousarray(((G2 + G2.T) / math.sqrt(2.0 * n)).astype(dt))
        del G2
    return out


def perturbations(n: int, nb: int, seed: int = 20210714, dtype=np.float64, decades: float = 1.0):
    """nb symmetric perturbations for the batched response (stand-ins for the Krylov vectors of PAPER.md:231):
    H1_b = 10^(-2 - decades * b) (G_b + G_b^T)/sqrt(2), G_b ~ N(0,1)^(n x n) -- magnitudes ``decades`` apart, so that a
    shared plane exponent would lose the small ones."""
    rng = np.random.default_rng(seed + 977)
    out = []
    for b in range(nb):
        G = rng.standard_normal((n, n))
        out.append(np.ascontiguousarray((10.0 ** (-2.0 - decades * b) * (G + G.T) / math.sqrt(2.0)).astype(dtype)))
        del G
    return out


def band_energy_closed_form(lam, n_occ):
    """sum of the n_occ lowest generator eigenvalues (what tr(DH) must equal
    for an exact-arithmetic H; a property of the INPUT, not of the method)."""
    return float(np.sort(np.asarray(lam, dtype=np.float64))[:n_occ].sum())


def ssh_chain(n: int, t1: float = 1.0, t2: float = 0.6, onsite: float = 0.0, dtype=np.float64):
    """A structured, SPARSE stand-in closer to the paper's tight-binding matrices than the dense
    Haar-rotated ones: the periodic dimerised chain (alternating hoppings t1, t2; n even), whose
    spectrum +-|t1 + t2 e^{ik}| has the gap 2|t1 - t2| at half filling and whose Gershgorin bounds
    +-(|t1| + |t2|) are TIGHT -- the regime in which the paper reports 14-16 layers.
    Returns (H, exact eigenvalues sorted ascending)."""
    if n % 2 or n < 4:
        raise ValueError("n must be even and >= 4")
    H = np.zeros((n, n), dtype=np.float64)
    idx = np.arange(n)
    hop = np.where(idx % 2 == 0, t1, t2)
    H[idx, (idx + 1) % n] = hop
    H[(idx + 1) % n, idx] = hop
    H[idx, idx] = onsite
    k = 2.0 * np.pi * np.arange(n // 2) / (n // 2)
    e = np.abs(t1 + t2 * np.exp(1j * k))
    lam = np.sort(np.concatenate([-e, e])) + onsite
    return np.ascontiguousarray(H.astype(dtype)), lam


def overlap_problem(n: int, n_occ: int, seed: int = 7, gap: float = 0.4):
    """A non-orthogonal stand-in: overlap S = I + 0.3 (B + B^T)/(2 sqrt n) (symmetric positive
    definite, well conditioned), its Loewdin inverse factor Z = S^(-1/2), and H = Z^-T (Q diag(lam) Q^T) Z^-1 so that
    the orthogonalised Hamiltonian Z^T H Z has the known, gapped spectrum lam.  Returns dict(H, S, Z, lam, Q)."""
    rng = np.random.default_rng(seed)
    B = rng.standard_normal((n, n))
    S = np.eye(n) + 0.3 * (B + B.T) / (2.0 * math.sqrt(n))
    w, V = np.linalg.eigh(S)
    assert w.min() > 0.2
    Z = (V / np.sqrt(w)) @ V.T                      # symmetric inverse square root
    Zinv = (V * np.sqrt(w)) @ V.T
    Q = _haar_q_numpy(rng.standard_normal((n, n)))
    lam = np.concatenate([rng.uniform(-1.0, -gap / 2, n_occ), rng.uniform(gap / 2, 1.0, n - n_occ)])
    Horth = (Q * lam) @ Q.T
    H = Zinv @ (0.5 * (Horth + Horth.T)) @ Zinv
    return dict(H=0.5 * (H + H.T), S=0.5 * (S + S.T), Z=0.5 * (Z + Z.T), lam=lam, Q=Q, n=n, n_occ=n_occ)


def hidden_eigenvector_problem(n: int, n_occ: int, hidden: float, orth_to, seed: int = 11, gap: float = 0.4):
    """Adversarial input for any Krylov spectral estimate started from the vector ``orth_to``: a gapped spectrum in
    [-1, 1] plus ONE outlier eigenvalue ``hidden`` (< -1: the lowest, occupied state; > 1: the highest, empty state) whose
    eigenvector is exactly orthogonal to ``orth_to``, so that in exact arithmetic the Krylov space never contains it.
    Returns (H, lam) with lam[k] the eigenvalue of column k of the (discarded) eigenvector matrix."""
    rng = np.random.default_rng(seed)
    v0 = np.asarray(orth_to, dtype=np.float64)
    v0 = v0 / np.linalg.norm(v0)
    q1 = rng.standard_normal(n)
    q1 -= (q1 @ v0) * v0
    q1 /= np.linalg.norm(q1)
    A = rng.standard_normal((n, n))
    A[:, 0] = q1
    Q, _ = np.linalg.qr(A)                          # column 0 = +-q1, the rest an orthonormal completion
    if hidden < 0:
        lam = np.concatenate([[hidden], rng.uniform(-1.0, -gap / 2, n_occ - 1), rng.uniform(gap / 2, 1.0, n - n_occ)])
    else:
        lam = np.concatenate([[hidden], rng.uniform(-1.0, -gap / 2, n_occ), rng.uniform(gap / 2, 1.0, n - n_occ - 1)])
    H = (Q * lam[None, :]) @ Q.T
    return np.ascontiguousarray(0.5 * (H + H.T)), lam
