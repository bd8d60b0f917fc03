"""CUDA-graph capture of the library calls: every device entry point only enqueues work on the caller's stream (kernels,
stream-ordered scratch from the library's memory pool, memsets), so a call -- or a whole right-hand side made of several
calls -- can be captured once and replayed without host work (B200 design rule: capture launch-bound inner loops in CUDA
graphs; the small configs are launch bound).  Replays must reproduce the eager results bit for bit."""
import numpy as np
import pytest

from paper_2412_13043_b200 import inputs

pytestmark = pytest.mark.gpu


def test_every_family_replays_bit_identically_from_a_cuda_graph():
    import torch
    from paper_2412_13043_b200 import binding as B
    up = lambda a: torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64)).cuda()
    rule = lambda r: tuple(up(a) for a in B.dfrg_quad_nodes(*r))
    calls, outs = [], []

    c = inputs.config1(0.2, n_field=300, n_q=33)
    rq, rho, u, du = rule(c["rule_q"]), up(c["rho"]), up(c["u"]), up(c["du"])
    flow, dchan = torch.empty_like(rho), torch.empty(2, rho.numel(), dtype=torch.float64, device="cuda")
    calls.append(lambda: B.dfrg_integrate_lpa(c["d"], c["T"], c["n_max"], c["reg_arg4d"], c["N"], c["prefactor"],
                                              c["reg_kind"], c["reg_order"], c["k"], rq, rho, u, du, flow, dchan=dchan))
    outs += [flow, dchan]

    c2 = inputs.config2(n_field=150, n_ext=5, n_q=37, n_c=8)
    r2q, r2c = rule(c2["rule_q"]), rule(c2["rule_c"])
    Z2, k2, m2, p2 = up(c2["Z"]), up(c2["coef"]), up(c2["m2"]), up(c2["pext"])
    o2 = torch.empty(5, 150, dtype=torch.float64, device="cuda")
    d2 = torch.empty_like(o2)
    calls.append(lambda: B.dfrg_integrate_loop4d(B.LOOP_TWOPOINT, c2["prefactor"], c2["reg_kind"], c2["reg_order"], c2["k"],
                                                 r2q, r2c, None, None, (Z2,), c2["lnq_lo"], c2["lnq_hi"], c2["interp"],
                                                 k2, m2, p2, o2, dout_dm2=d2))
    outs += [o2, d2]

    c3 = inputs.config3(n_p=3, n_alpha=2, n_q=16, n_c1=8, n_c2=4)
    r3 = {ax: rule(c3["rule_" + ax]) for ax in ("q", "c1", "c2", "phi")}
    t3 = (up(c3["ZA"]), up(c3["Zc"]), up(c3["L3"]))
    k3, e3 = up(c3["coef"]), up(c3["ext"])
    o3 = torch.empty(e3.shape[0], dtype=torch.float64, device="cuda")
    calls.append(lambda: B.dfrg_integrate_loop4d(B.LOOP_THREEPOINT, c3["prefactor"], c3["reg_kind"], c3["reg_order"],
                                                 c3["k"], r3["q"], r3["c1"], r3["c2"], r3["phi"], t3, c3["lnq_lo"],
                                                 c3["lnq_hi"], c3["interp"], k3, None, e3, o3,
                                                 ext_outer=c3["ext_outer"]))
    outs.append(o3)

    c4 = inputs.config4(n_field=300, n_p=2, n_jext=3, n_q=9, n_c=8)
    c4["n_max"] = 3
    r4q, r4c = rule(c4["rule_q"]), rule(c4["rule_c"])
    a4 = [up(c4[k_]) for k_ in ("Zpsi", "Zphi", "coef", "m2psi", "m2phi", "pext")]
    o4 = [torch.empty(2, 3, 300, dtype=torch.float64, device="cuda") for _ in range(3)]
    calls.append(lambda: B.dfrg_integrate_matsubara3d(c4["T"], c4["n_max"], c4["prefactor"], c4["reg_kind"],
                                                      c4["reg_order"], c4["k"], r4q, r4c, a4[0], a4[1], c4["lnq_lo"],
                                                      c4["lnq_hi"], c4["interp"], a4[2], a4[3], a4[4], a4[5], 3, o4[0],
                                                      o4[1], reg_arg4d=0, mu=0.3, out_im=o4[2]))
    outs += o4

    def whole_rhs():
        for f in calls:
            f()

    whole_rhs()                                   # eager (also warms the library's memory pool up)
    torch.cuda.synchronize()
    ref = [o.clone() for o in outs]
    for o in outs:
        o.fill_(float("nan"))
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        whole_rhs()                               # captured: nothing runs yet
    for _ in range(3):
        g.replay()
    torch.cuda.synchronize()
    for o, r in zip(outs, ref):
        assert torch.equal(o, r) or (torch.isnan(o) == torch.isnan(r)).all() and torch.equal(torch.nan_to_num(o), torch.nan_to_num(r))
    # new inputs in the same buffers, same graph: the replay sees them
    rho.mul_(0.5)
    u.add_(0.25)
    g.replay()
    torch.cuda.synchronize()
    graph_flow = flow.clone()
    calls[0]()
    torch.cuda.synchronize()
    assert torch.equal(graph_flow, flow) and not torch.equal(flow, ref[0])
