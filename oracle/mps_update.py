"""oracle.mps_update - TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).

Plain CPU definition of the minimal MPS two-site update ("nested Schmidt decomposition",
PAPER.md:39 "Hermitian matrix diagonalization ... the dominant factor", PAPER.md:35 the epsilon ~ 2^(-n+1) example), written
out index by index in mpmath at prec + 128 bits, with the Hermitian eigendecomposition taken from the pinned MPFR Jacobi oracle:

    Theta0[(a,i),(j,c)] = sum_k L[(a,i),k] R[k,(j,c)]
    Theta[(a,i'),(j',c)] = sum_{i,j} G[(i'j'),(ij)] Theta0[(a,i),(j,c)]
    rho = Theta Theta^H ;  rho = U diag(w) U^H (oracle.diag_herm on rho rounded to prec bits) ;  R' = U^H Theta
    weights descending; kept = #{w_k > 2^-cutoff_bits trace(rho)}

Parity status: pinned (tests/test_oracle_mps_pins.py: product state, Bell pair from CNOT, the paper's epsilon example with
weights known by construction, trace identity, weights = squared singular values by the pinned SVD oracle)."""
from __future__ import annotations

import numpy as np

import oracle
import zkd_inputs as zi


def _to_mp(mp, buf, R, C, prec):
    rb = zi.real_bytes(prec)
    flat = np.asarray(buf).reshape(R, C, 2, rb)
    M = mp.matrix(R, C)
    for i in range(R):
        for j in range(C):
            M[i, j] = mp.mpc(zi.to_mpf(flat[i, j, 0], prec), zi.to_mpf(flat[i, j, 1], prec))
    return M


def _from_mp(mp, M, prec):
    rb = zi.real_bytes(prec)
    out = np.zeros((M.rows, M.cols, 2, rb), dtype=np.uint8)
    for i in range(M.rows):
        for j in range(M.cols):
            z = mp.mpc(M[i, j])
            out[i, j, 0] = np.frombuffer(zi.from_mpf(z.real, prec), dtype=np.uint8)
            out[i, j, 1] = np.frombuffer(zi.from_mpf(z.imag, prec), dtype=np.uint8)
    return out.reshape(-1)


def theta(mp, L, R, G, chiL, chiC, chiR, d, prec):
    mL, mR = chiL * d, d * chiR
    Lm, Rm, Gm = _to_mp(mp, L, mL, chiC, prec), _to_mp(mp, R, chiC, mR, prec), _to_mp(mp, G, d * d, d * d, prec)
    T0 = mp.matrix(mL, mR)
    for r in range(mL):
        for c in range(mR):
            T0[r, c] = sum(Lm[r, k] * Rm[k, c] for k in range(chiC))
    T = mp.matrix(mL, mR)
    for a in range(chiL):
        for ip in range(d):
            for jp in range(d):
                for c in range(chiR):
                    T[a * d + ip, jp * chiR + c] = sum(Gm[ip * d + jp, i * d + j] * T0[a * d + i, j * chiR + c]
                                                       for i in range(d) for j in range(d))
    return T


def two_site_update(mp, L, R, G, chiL, chiC, chiR, d, cutoff_bits=700, prec=768):
    """Returns dict(weights=[mpf] descending, Lnew=mp.matrix (mL x mL), Rnew=mp.matrix (mL x mR), theta=mp.matrix, kept=int,
    rho_api=uint8 array)."""
    old = mp.mp.prec
    mp.mp.prec = prec + 128
    try:
        mL, mR = chiL * d, d * chiR
        T = theta(mp, L, R, G, chiL, chiC, chiR, d, prec)
        rho = mp.matrix(mL, mL)
        for r in range(mL):
            for c in range(mL):
                rho[r, c] = sum(T[r, k] * mp.conj(T[c, k]) for k in range(mR))
        rho_api = _from_mp(mp, rho, prec)
        lam, X, info = oracle.diag_herm(rho_api, mL, prec=prec)
        assert info["status"] == 0
        lam_m = zi.rvector_to_mp(lam, mL, prec)
        Xm = zi.cmatrix_to_mp(X, mL, prec)
        w = [lam_m[mL - 1 - k] for k in range(mL)]
        Ln = mp.matrix(mL, mL)
        for r in range(mL):
            for k in range(mL):
                Ln[r, k] = Xm[r, mL - 1 - k]
        Rn = mp.matrix(mL, mR)
        for k in range(mL):
            for c in range(mR):
                Rn[k, c] = sum(mp.conj(Ln[r, k]) * T[r, c] for r in range(mL))
        tr = sum(rho[r, r].real for r in range(mL))
        kept = sum(1 for x in w if x > mp.ldexp(tr, -cutoff_bits))
        return {"weights": w, "Lnew": Ln, "Rnew": Rn, "theta": T, "kept": kept, "rho_api": rho_api, "trace": tr}
    finally:
        mp.mp.prec = old
