"""GPU parity of the closed-shell entry gfcc_create_closed_shell (the paper's production runs are closed-shell and
handle the alpha electrons): spatial tensors in, device-side expansion, ordinary spin-orbital handle out.  The oracle side is
oracle.closed_shell.expand_closed_shell (pinned against the spin-free Fock-space definition) + the spin-orbital oracle.  -m gpu."""
import numpy as np
import pytest
import torch

import oracle
from oracle.closed_shell import expand_closed_shell, so_index
from gfcc_testutil import random_x, relmax
from test_oracle_closed_shell import spatial_system

pytestmark = pytest.mark.gpu


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("no,nv,Q", [(1, 1, 1), (2, 3, 4), (3, 5, 6), (4, 9, 12)])
def test_closed_shell_handle_equals_oracle_on_expanded_tensors(no, nv, Q):
    import paper_2010_04768_b200 as g
    s = spatial_system(no, nv, Q, seed=3 * no + nv)
    x = expand_closed_shell(no, nv, s["fock"], s["T1"], s["T2"], s["L1"], s["L2"], s["Lchol"])
    o, v = x["o"], x["v"]
    orc = oracle.Oracle(o, v, Q, x["fock"], x["T1"], x["T2p"], x["L1"], x["L2p"], x["Lchol"], oracle.MODE_DEF | oracle.MODE_EA)
    h = g.gfcc_create_closed_shell(no, nv, Q, *[dev(s[k]) for k in ("fock", "T1", "T2", "L1", "L2", "Lchol")])
    for name in ("Fme", "Fmi", "Fae"):
        ref = orc.get(name)
        assert relmax(g.gfcc_get_intermediate(h, name).cpu().numpy().reshape(ref.shape), ref) < 1e-12, name
    x1, x2 = random_x(o, v, 3, seed=2)
    w = np.array([-0.4, -0.7, 0.2])
    S1, S2 = orc.sigma(w, 0.02, x1, x2)
    G1, G2 = g.gfcc_sigma_ip(h, w, 0.02, dev(x1), dev(x2))
    assert relmax(G1.cpu().numpy(), S1) < 1e-10 and relmax(G2.cpu().numpy(), S2) < 1e-10
    # closed-shell G for alpha targets: IP and EA parts, against dense LU on the expanded tensors
    alpha = [so_index(no, nv, p, 0) for p in range(no + nv)]
    beta = [so_index(no, nv, p, 1) for p in range(no + nv)]
    ws = [-0.35, 0.45]
    ndim = max(o + o * (o - 1) // 2 * v, v + o * v * (v - 1) // 2)
    g.gfcc_set_option(h, "gmres_m", ndim + 2)          # full GMRES: the random couplings put poles inside the omega range
    g.gfcc_set_option(h, "gmres_maxit", 4 * ndim)
    G = g.gfcc_solve_ip(h, alpha + beta, ws, 0.03, 1e-11)
    Gd = orc.G_dense(alpha + beta, ws, 0.03)
    assert relmax(G, Gd) < 1e-8
    k = len(alpha)
    scale = np.abs(G).max()
    assert np.abs(G[:, :k, :k] - G[:, k:, k:]).max() < 1e-8 * scale          # G_{p alpha, q alpha} = G_{p beta, q beta}
    assert np.abs(G[:, :k, k:]).max() < 1e-8 * scale                          # mixed-spin elements vanish
    GA = g.gfcc_solve_ea(h, alpha, ws, 0.03, 1e-11)
    assert relmax(GA, orc.G_dense_ea(alpha, ws, 0.03)) < 1e-8
    g.gfcc_destroy(h)
