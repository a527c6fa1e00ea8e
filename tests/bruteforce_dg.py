"""Brute-force dense numpy DG operator on tiny FLAT brick meshes -- an independent transcription of the
paper's equations used only to pin the oracle (tests/test_oracle_dg.py).

Differences from oracle/dg_oracle.cpp on purpose: strong form (eq. 32) instead of weak; dense
Np x Np Kronecker derivative matrices instead of sum factorisation; Lagrange derivatives from numpy.poly1d;
structure-of-arrays numpy state; plain p - p_r instead of the R12 difference formula; closed-form axis
aligned geometry (Delta, normals, lift) instead of metric terms.
"""
import numpy as np

import workloads as W


def lgl_weights(xi):
    from numpy.polynomial import legendre as L
    N = xi.size - 1
    c = np.zeros(N + 1); c[N] = 1.0
    return 2.0 / (N * (N + 1) * L.legval(xi, c) ** 2)


def lagrange_derivative_matrix(xi):
    Nq = xi.size
    D = np.zeros((Nq, Nq))
    for j in range(Nq):
        others = np.delete(xi, j)
        Lj = np.poly1d(others, r=True) / np.prod(xi[j] - others)
        D[:, j] = Lj.deriv()(xi)
    return D


class BruteDG:
    def __init__(self, cfg):
        assert cfg.get("geom", 0) == 0
        self.cfg = cfg
        self.N = cfg["N"]; self.Nq = Nq = self.N + 1; self.Np = Nq ** 3
        self.ne = cfg["ne"]; self.Ne = int(np.prod(self.ne))
        self.nvar = cfg["nvar"]
        self.xi = W.lgl_nodes(self.N)
        self.w = lgl_weights(self.xi)
        D = lagrange_derivative_matrix(self.xi)
        I = np.eye(Nq)
        self.h = [(cfg["hi"][d] - cfg["lo"][d]) / self.ne[d] for d in range(3)]
        # physical derivative matrices on one element (node n = i + Nq j + Nq^2 k)
        self.Dx = [(2 / self.h[0]) * np.kron(I, np.kron(I, D)),
                   (2 / self.h[1]) * np.kron(I, np.kron(D, I)),
                   (2 / self.h[2]) * np.kron(D, np.kron(I, I))]
        self.z = W.node_coords(cfg)[..., 2]
        self.Delta = (self.h[0] * self.h[1] * self.h[2]) ** (1.0 / 3.0) / self.N
        n = np.arange(self.Np)
        self.ijk = np.stack([n % Nq, (n // Nq) % Nq, n // (Nq * Nq)], axis=1)

    # -- thermodynamics, vectorised over nodes
    def prim(self, Q, z, ref=None):
        c = self.cfg
        rho = Q[..., 0]; u = Q[..., 1:4] / rho[..., None]
        q = Q[..., 5] / rho if self.nvar == 6 else np.zeros_like(rho)
        cvm = c["c_vd"] * (1 - q) + c["c_vv"] * q
        Rm = c["R_d"] * (1 - q) + c["R_v"] * q
        eint = Q[..., 4] / rho - 0.5 * (u ** 2).sum(-1) - c["grav"] * z
        T = c["T_0"] + (eint - q * c["I_v0"]) / cvm
        p = rho * Rm * T
        out = dict(rho=rho, u=u, q=q, T=T, p=p, h=(Q[..., 4] + p) / rho, c=np.sqrt((1 + Rm / cvm) * Rm * T))
        if ref is not None:
            out["pp"] = p - ref["p"]; out["rho_r"] = ref["rho"]
        else:
            out["pp"] = p; out["rho_r"] = np.zeros_like(rho)
        return out

    def ref_state(self):
        c = self.cfg
        if not c.get("use_ref"):
            return None
        Qr = np.zeros((self.Ne, self.Np, self.nvar))
        Qr[..., 0] = c["ref_rho"]; Qr[..., 4] = c["ref_rhoe"]
        if self.nvar == 6:
            Qr[..., 5] = c["ref_rhoq"]
        return dict(rho=Qr[..., 0], p=self.prim(Qr, self.z)["p"])

    def neighbour(self, e, f):
        Ex, Ey, Ez = self.ne
        ec = [e % Ex, (e // Ex) % Ey, e // (Ex * Ey)]
        d = f // 2; ec[d] += 1 if f % 2 else -1
        if ec[d] < 0 or ec[d] >= self.ne[d]:
            if self.cfg["bc"][d]:
                return -1
            ec[d] %= self.ne[d]
        return ec[0] + Ex * (ec[1] + Ey * ec[2])

    def face_nodes(self, f):
        d = f // 2; at = self.N if f % 2 else 0
        mine = np.where(self.ijk[:, d] == at)[0]
        theirs = mine + (-(self.N) if f % 2 else self.N) * (self.Nq ** d)
        return mine, theirs

    def grad_vars(self, P):
        return np.concatenate([P["u"], P["h"][..., None], P["q"][..., None]], axis=-1)   # [.., 5]

    def gradient(self, Q):
        ref = self.ref_state()
        P = self.prim(Q, self.z, ref)
        s = self.grad_vars(P)                                   # [Ne, Np, 5]
        G = np.zeros((self.Ne, self.Np, 5, 3))
        for e in range(self.Ne):
            for d in range(3):
                G[e, :, :, d] = self.Dx[d] @ s[e]
            for f in range(6):
                d = f // 2; sgn = 1.0 if f % 2 else -1.0
                mine, theirs = self.face_nodes(f)
                en = self.neighbour(e, f)
                lift = (2 / self.h[d]) / self.w[0]
                sm = s[e, mine]
                if en >= 0:
                    sstar = 0.5 * (sm + s[en, theirs])
                else:
                    sstar = sm.copy(); sstar[:, d] = 0.0          # u_bc = u - (n.u) n for an axis-aligned wall
                G[e, mine, :, d] += lift * sgn * (sstar - sm)
        return G

    def fluxes(self, Q, P, G):
        """Total physical flux F[..., v, c] = F1 + F2."""
        c = self.cfg; nv = self.nvar
        rho, u = P["rho"], P["u"]
        F = np.zeros(Q.shape[:-1] + (nv, 3))
        for cc in range(3):
            F[..., 0, cc] = Q[..., 1 + cc]
            for i in range(3):
                F[..., 1 + i, cc] = Q[..., 1 + i] * u[..., cc] + (P["pp"] if i == cc else 0.0)
            F[..., 4, cc] = (Q[..., 4] + P["p"]) * u[..., cc]
            if nv == 6:
                F[..., 5, cc] = Q[..., 5] * u[..., cc]
        if c["sgs"]:
            gu = G[..., 0:3, :]                                   # d u_i / d x_j
            S = 0.5 * (gu + np.swapaxes(gu, -1, -2))
            nu = (c["C_s"] * self.Delta) ** 2 * np.sqrt(2 * (S ** 2).sum((-1, -2)))
            Dt = nu / c["Pr_t"]
            tau = -2 * nu[..., None, None] * S
            dq = -Dt[..., None] * G[..., 4, :] if nv == 6 else np.zeros_like(G[..., 4, :])
            JD = -Dt[..., None] * G[..., 3, :]
            F[..., 0, :] += rho[..., None] * dq
            F[..., 1:4, :] += rho[..., None, None] * tau + Q[..., 1:4, None] * dq[..., None, :]
            F[..., 4, :] += rho[..., None] * np.einsum("...cj,...j->...c", tau, u) + rho[..., None] * JD
            if nv == 6:
                F[..., 5, :] += rho[..., None] * dq
        return F

    def rhs(self, Q):
        c = self.cfg; nv = self.nvar
        ref = self.ref_state()
        P = self.prim(Q, self.z, ref)
        G = self.gradient(Q) if c["sgs"] else np.zeros((self.Ne, self.Np, 5, 3))
        F = self.fluxes(Q, P, G)
        dQ = np.zeros_like(Q)
        for e in range(self.Ne):
            for d in range(3):
                dQ[e] -= self.Dx[d] @ F[e, :, :, d]
            dQ[e, :, 3] -= (P["rho"][e] - P["rho_r"][e]) * c["grav"]
            for f in range(6):
                d = f // 2; sgn = 1.0 if f % 2 else -1.0
                mine, theirs = self.face_nodes(f)
                en = self.neighbour(e, f)
                lift = (2 / self.h[d]) / self.w[0]
                Ym = Q[e, mine]
                nFm = sgn * F[e, mine, :, d]                        # n . F_total^-
                um = sgn * P["u"][e, mine, d]; cm = P["c"][e, mine]
                if en >= 0:
                    Yp = Q[en, theirs]
                    nFp = sgn * F[en, theirs, :, d]
                    lam = np.maximum(np.abs(um) + cm, np.abs(sgn * P["u"][en, theirs, d]) + P["c"][en, theirs])
                    Fstar = 0.5 * (nFm + nFp) + 0.5 * lam[:, None] * (Ym - Yp)
                else:
                    # mirror ghost: the Rusanov flux of (Y-, mirror) evaluated from its definition
                    Yp = Ym.copy(); Yp[:, 1 + d] = -Ym[:, 1 + d]
                    Pm = {k: (v[e, mine] if isinstance(v, np.ndarray) else v) for k, v in P.items()}
                    Pp = dict(Pm); Pp["u"] = Pm["u"].copy(); Pp["u"][:, d] *= -1
                    Gz = np.zeros((mine.size, 5, 3))
                    sg, c["sgs"] = c["sgs"], 0
                    F1m = self.fluxes(Ym, Pm, Gz); F1p = self.fluxes(Yp, Pp, Gz)
                    c["sgs"] = sg
                    lam = np.abs(um) + cm
                    Fstar = 0.5 * sgn * (F1m[:, :, d] + F1p[:, :, d]) + 0.5 * lam[:, None] * (Ym - Yp)
                    if f == 4 and c["shf_bottom"]:
                        Fstar[:, 4] += -c["shf_bottom"]
                dQ[e, mine] += lift * (nFm - Fstar)
        return dQ
