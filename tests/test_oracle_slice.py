"""The identity behind the render path's time slice (dash_hash4d_slice_t + dash_hash4d_slice_fwd; Q29),
checked against the 4D oracle on the CPU: for ONE timestamp t the quadrilinear interpolation of Eq. 9 factors into a
per-level blend of the two t-layers followed by a trilinear lookup,
    B_l[u] = (1 - w_t) table_l[u XOR a] + w_t table_l[u XOR b],  a = (c_t pi_4) mod T,  b = ((c_t + 1) pi_4) mod T
    out = trilinear lookup of B_l at slot (g_x pi_1 XOR g_y pi_2 XOR g_z pi_3) mod T
which holds because for a power-of-two T the "mod T" of Eq. 8 keeps the low bits and so commutes with XOR; on a dense
level the blend is over the vertex layers g_t = c_t, c_t + 1 and the slot is g_x + S(g_y + S g_z)."""
import numpy as np
import pytest

import oracle
from dash_inputs import make_queries_uniform

PI = (1, 2654435761, 805459861, 3674653429)


def slice_then_trilinear(xyz, t, table, res_s, res_t, dense, T):
    L, _, F = table.shape
    out = np.zeros((len(xyz), L * F))
    for l in range(L):
        ns, nt = int(res_s[l]), int(res_t[l])
        ct, wt = oracle.oracle_locate(float(t), nt)
        tab = table[l].astype(np.float64)
        if dense[l]:
            S = ns + 1
            B = (1 - wt) * tab[S ** 3 * ct: S ** 3 * (ct + 1)] + wt * tab[S ** 3 * (ct + 1): S ** 3 * (ct + 2)]
        else:
            a, b = (ct * PI[3]) % 2 ** 32 % T, ((ct + 1) * PI[3]) % 2 ** 32 % T
            u = np.arange(T)
            B = (1 - wt) * tab[u ^ a] + wt * tab[u ^ b]
        for n, p in enumerate(xyz):
            cw = [oracle.oracle_locate(float(p[d]), ns) for d in range(3)]
            for k in range(8):
                g = [cw[d][0] + ((k >> d) & 1) for d in range(3)]
                w = np.prod([cw[d][1] if (k >> d) & 1 else 1 - cw[d][1] for d in range(3)])
                if dense[l]:
                    s = g[0] + (ns + 1) * (g[1] + (ns + 1) * g[2])
                else:
                    s = (((g[0] * PI[0]) ^ (g[1] * PI[1]) ^ (g[2] * PI[2])) & 0xFFFFFFFF) % T
                out[n, l * F:(l + 1) * F] += w * B[s]
    return out


@pytest.mark.parametrize("dense_coarse", [True, False])
@pytest.mark.parametrize("tval", [0.0, 0.37, 0.5, float(np.float32(1) - np.float32(2.0 ** -24))])
def test_slice_identity_matches_4d_oracle(dense_coarse, tval):
    L, F, T = 6, 2, 1 << 12
    cfg = oracle.make_config(L, F, T, 4, 200, 2, 40, dense_coarse=dense_coarse)
    rs, rt, dn = oracle.oracle_resolutions(cfg)
    assert (dn[0] and not dn[-1]) if dense_coarse else not dn.any()
    xyz, _ = make_queries_uniform(21, 60)
    xyz[0] = [0.0, 1.0, 0.999]
    table = np.random.default_rng(1).uniform(-1, 1, (L, T, F)).astype(np.float32)
    t = np.array([tval], np.float32)
    want = oracle.oracle_fwd(cfg, 60, xyz, t, table, t_stride=0).astype(np.float64)
    got = slice_then_trilinear(xyz, t[0], table, rs, rt, dn, T)
    np.testing.assert_allclose(got, want, rtol=0, atol=2e-7)


def test_xor_does_not_commute_with_mod_for_other_table_sizes():
    """Why the slice needs a power-of-two T on hashed levels (the library returns UNSUPPORTED otherwise)."""
    T = 100003
    u, a = (5 * PI[1]) % 2 ** 32, (3 * PI[3]) % 2 ** 32
    assert (u ^ a) % T != (u % T) ^ (a % T)
