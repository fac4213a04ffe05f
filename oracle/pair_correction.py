"""pair_correction.py -- fp64 ORACLE of the short-range pair correction.  TEST INFRASTRUCTURE ONLY.

P:105: "TorchNEP fully supports the Ziegler-Biersack-Littmark (ZBL) potential [24] as a short-range correction".
The paper prints neither the screening function's constants nor the radii between which the correction is switched off
(Ref. [24] and Fig. S1 are not part of PAPER.md), so nothing of the kind is stored here or in the CUDA library: the term has a
FIXED FORM, a screened Coulomb repulsion, and every number in it is an argument (reading G29):

    E_corr = sum over undirected pairs {(i,0), (j,n)} with r < r_outer of  phi_ij(r),
    phi_ij(r) = sw(r) * (k_C Z_i Z_j / r) * sum_m coef_m exp(-expo_m r / a_ij),      a_ij = a_prefac / (Z_i^a_pow + Z_j^a_pow),
    sw(r) = 1 (r <= r_inner);  1/2 (1 + cos(pi (r - r_inner) / (r_outer - r_inner))) (r_inner < r < r_outer);  0 beyond,

with k_C = e^2 / (4 pi eps_0) in eV Angstrom (also the caller's).  It depends on no parameter of the model: it adds to E, F and W
and contributes nothing to grad_theta L.  Forces and virial are its derivatives: F_i = -dE_corr/dr_i, W = -sum d (x) dE/dd.

Plain numpy over the radial neighbour list of oracle.nep_oracle.OracleData (every directed pair i -> (j, n), so every undirected
pair appears twice and carries half of phi each time); no blocking, no shared code with paper_2606_19557_b200/.
Pins: tests/test_oracle_pair.py (Coulomb's law in the unscreened limit, the screening slope, the switch at its mid-point and at
r_outer, forces and virial against finite differences of E, sum F = 0, no dependence on theta).
"""
import numpy as np


def switch(r, r_inner, r_outer):
    """sw(r) and d sw / d r (reading G29: cosine switch, the same shape as the cutoff function of Eq. 18)."""
    r = np.asarray(r, np.float64)
    t = (r - r_inner) / (r_outer - r_inner)
    mid = (r > r_inner) & (r < r_outer)
    sw = np.where(r <= r_inner, 1.0, 0.0)
    dsw = np.zeros_like(r)
    sw = np.where(mid, 0.5 * (1.0 + np.cos(np.pi * t)), sw)
    dsw = np.where(mid, -0.5 * np.pi / (r_outer - r_inner) * np.sin(np.pi * t), dsw)
    return sw, dsw


def pair_energy(r, Zi, Zj, r_inner, r_outer, coef, expo, a_prefac, a_pow, coulomb_k):
    """phi_ij(r) and d phi / d r for arrays r, Zi, Zj."""
    r = np.asarray(r, np.float64)
    a = a_prefac / (np.power(Zi, a_pow) + np.power(Zj, a_pow))
    x = r / a
    scr = np.zeros_like(r)
    dscr = np.zeros_like(r)
    for c, e in zip(coef, expo):
        scr = scr + c * np.exp(-e * x)
        dscr = dscr - c * e / a * np.exp(-e * x)
    coul = coulomb_k * Zi * Zj / r
    dcoul = -coul / r
    sw, dsw = switch(r, r_inner, r_outer)
    phi0 = coul * scr
    dphi0 = dcoul * scr + coul * dscr
    return sw * phi0, dsw * phi0 + sw * dphi0


def pair_correction(data, Z, r_inner, r_outer, coef, expo, a_prefac, a_pow, coulomb_k):
    """E [S], F [N, 3], W [S, 9] of the correction for every structure of `data` (an OracleData; r_outer <= its radial cutoff)."""
    assert 0.0 <= r_inner < r_outer <= data.model.rc_R
    Z = np.asarray(Z, np.float64)
    coef = np.asarray(coef, np.float64); expo = np.asarray(expo, np.float64)
    S, N = data.n_struct, data.n_atoms_total
    E = np.zeros(S); F = np.zeros((N, 3)); W = np.zeros((S, 9))
    n_per = np.diff(data.atom_off)
    s_of_atom = np.repeat(np.arange(S), n_per)
    deg = np.diff(data.offR)
    i = np.repeat(np.arange(N), deg)                       # first atom of every directed pair
    if len(i) == 0:
        return E, F, W
    s = s_of_atom[i]
    j = data.atom_off[s] + data.jR                         # global index of the neighbour
    box = data.box[s].reshape(-1, 3, 3)                    # rows a, b, c
    sh = data.shR.astype(np.float64)
    # C1: d = (((r_j - r_i) + n_a a) + n_b b) + n_c c
    d = (((data.pos[j] - data.pos[i]) + sh[:, 0:1] * box[:, 0]) + sh[:, 1:2] * box[:, 1]) + sh[:, 2:3] * box[:, 2]
    r = np.sqrt(np.sum(d * d, axis=1))
    inside = r < r_outer
    i, j, s, d, r = i[inside], j[inside], s[inside], d[inside], r[inside]
    phi, dphi = pair_energy(r, Z[data.type[i]], Z[data.type[j]], r_inner, r_outer, coef, expo, a_prefac, a_pow, coulomb_k)
    # every undirected pair is listed twice: half of phi per listing
    np.add.at(E, s, 0.5 * phi)
    # E depends on r_i through d of the listing i -> j (d = .. - r_i) and of the listing j -> i (d = r_i - ..): both give the same
    # term, so F_i = -dE/dr_i = sum over the listings i -> j of phi'(r) d / r
    np.add.at(F, i, (dphi / r)[:, None] * d)
    # W = -sum over listings of d (x) d(phi / 2)/dd
    dEdd = (0.5 * dphi / r)[:, None] * d
    np.add.at(W, s, -(d[:, :, None] * dEdd[:, None, :]).reshape(-1, 9))
    return E, F, W
