"""Domain decomposition with halo exchange.

CPU (world_size 2 and 3 over gloo): the partitioner's invariants, and the oracle run rank by rank on the split case with a real
point-to-point exchange of U_f and G_f, against the oracle on the whole case.
GPU (-m gpu, one device): the library's partitioned right-hand side (fr_rhs_phase + halo buffers), the ranks' phases launched one
after the other with device copies standing in for the transport, against the single-context right-hand side bit for bit.
"""
import os
import sys

import numpy as np
import pytest

from fr_inputs import cases, partition as P
from util import field_errors, oracle_rhs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _case(kind):
    if kind == "box":
        return cases.config2(4, 2, "ns", numbering="random", ldg_beta=0.3, ldg_tau=0.1)
    return cases.config3(p=2, ntheta=16, nz=4, nlayers=4, nr=4, numbering="random")


def test_partition_weights_and_split_invariants():
    case = _case("cyl")
    for nparts in (2, 3, 4):
        part = P.partition(case, nparts)
        w = np.zeros(nparts)
        for t, pt in zip(case["etypes"], part):
            w += np.bincount(pt, minlength=nparts) * P.WEIGHT[t]
        assert w.max() / w.mean() < 1.05                       # weighted balance (hex : pri : tet = 3 : 2 : 1)
        subs, maps = P.split_case(case, part)
        # every element on exactly one rank; every flux point of a rank in exactly one pair or boundary list
        for t, e in enumerate(case["eles"]):
            ids = np.concatenate([g for mp in maps for (tt, g) in mp if tt == t])
            assert np.array_equal(np.sort(ids), np.arange(e["neles"]))
        ncut = 0
        for r, s in enumerate(subs):
            gt = len(s["eles"])
            seen = [np.zeros((e["nfpts"], e["neles"]), dtype=int) for e in s["eles"]]
            for side in ("l", "r"):
                for t in range(gt):
                    m = s["ifc"][side + "_et"] == t
                    np.add.at(seen[t], (s["ifc"][side + "_fpt"][m], s["ifc"][side + "_ele"][m]), 1)
            for b in s["bcs"]:
                for t in range(gt):
                    m = b["et"] == t
                    np.add.at(seen[t], (b["fpt"][m], b["ele"][m]), 1)
            assert all(np.all(x == 1) for x in seen)
            gl, gr = s["ifc"]["l_et"] == gt, s["ifc"]["r_et"] == gt
            assert not np.any(gl & gr)
            g = np.concatenate([s["ifc"]["l_ele"][gl], s["ifc"]["r_ele"][gr]])
            assert np.array_equal(np.sort(g), np.arange(s["halo"]["nghost"]))      # every ghost referenced exactly once
            assert sum(p_["count"] for p_ in s["halo"]["peers"]) == s["halo"]["nghost"]
            ncut += s["halo"]["nghost"]
            # send counts are symmetric
            for p_ in s["halo"]["peers"]:
                back = [q for q in subs[p_["rank"]]["halo"]["peers"] if q["rank"] == r]
                assert len(back) == 1 and back[0]["count"] == p_["count"]
        assert ncut % 2 == 0 and ncut > 0


def _oracle_worker(rank, world, port, kind, q):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from oracle import fr_oracle as O
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    case = _case(kind)
    subs, maps = P.split_case(case, P.partition(case, world))
    s = subs[rank]
    h = s["halo"]

    def exchange(name, own):
        # own [V, n_send] in the peers' ghost order; returns [V, n_ghost]
        out = np.empty_like(own)
        ops, keep = [], []
        for p_ in h["peers"]:
            sl = slice(p_["start"], p_["start"] + p_["count"])
            snd = torch.from_numpy(np.ascontiguousarray(own[:, sl]))
            rcv = torch.empty_like(snd)
            keep.append((sl, rcv))
            ops += [dist.P2POp(dist.isend, snd, p_["rank"]), dist.P2POp(dist.irecv, rcv, p_["rank"])]
        for w in dist.batch_isend_irecv(ops):
            w.wait()
        for sl, rcv in keep:
            out[:, sl] = rcv.numpy()
        return out

    got = O.rhs(s["cfg"], s["eles"], s["ifc"], s["bcs"], s["u0"], halo=dict(et=h["et"], fpt=h["fpt"], ele=h["ele"], exchange=exchange))
    q.put((rank, got))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("kind,world", [("box", 2), ("cyl", 2), ("cyl", 3)])
def test_partitioned_oracle_equals_whole_domain_oracle_gloo(kind, world):
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() * 7 + world * 13 + len(kind)) % 2000
    procs = [ctx.Process(target=_oracle_worker, args=(r, world, port, kind, q)) for r in range(world)]
    for p_ in procs:
        p_.start()
    res = dict(q.get(timeout=300) for _ in range(world))
    for p_ in procs:
        p_.join(timeout=60)
        assert p_.exitcode == 0
    case = _case(kind)
    _, maps = P.split_case(case, P.partition(case, world))
    got = P.assemble(case, maps, [res[r] for r in range(world)])
    ref = oracle_rhs(case)
    assert all(np.isfinite(g).all() for g in got)
    err, _ = field_errors(got, ref)
    assert err.max() < 1e-12, err


# ---------------------------------------------------------------------------- the library's partitioned path, one device
@pytest.mark.gpu
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("kind,world", [("box", 2), ("cyl", 2), ("cyl", 3)])
def test_partitioned_gpu_rhs_and_step_equal_single_context_bitwise(kind, world, prec):
    """Every rank's part as its own context on the one device; the ranks' phases are launched one after the other and device
    copies stand in for the NCCL transfers (paper_1409_0405_b200.halo.local_exchange).  The assembled right-hand side and the
    state after one RK45[2R+] step must equal the single-context results bit for bit (the arithmetic per column and per
    flux-point pair is the same; only where the data lives differs), and the oracle within the parity tolerance."""
    import torch
    from gpu_util import gpu_rhs, round_case_to_f32, to_device
    from paper_1409_0405_b200 import Context, halo as H
    case = _case(kind)
    whole = Context(case, prec=prec, stepper="rk45")
    got_whole, _ = gpu_rhs(whole, case["u0"])
    dt = 1e-4 if kind == "box" else 1e-6
    whole.set_state(case["u0"])
    whole.rk_step(dt)
    st_whole = whole.get_state()
    assert all(np.isfinite(x).all() for x in st_whole)
    whole.close()
    subs, maps = P.split_case(case, P.partition(case, world))
    ctxs = [Context(s, prec=prec, stepper="rk45") for s in subs]
    xchs = [H.HaloExchange(c) for c in ctxs]
    d_u = [to_device(c, s["u0"]) for c, s in zip(ctxs, subs)]
    d_out = [[torch.full_like(t, float("nan")) for t in du] for du in d_u]
    up = [[t.data_ptr() for t in du] for du in d_u]
    op = [[t.data_ptr() for t in do] for do in d_out]
    for ph in range(3):
        for c, u, o in zip(ctxs, up, op):
            c.rhs_phase(ph, u, o if ph == 2 else None)
        torch.cuda.synchronize()
        if ph < 2:
            H.local_exchange(xchs, ph)
            torch.cuda.synchronize()
    parts = [[t.cpu().numpy().astype(np.float64)[:, :, :u.shape[2]] for t, u in zip(do, s["u0"])] for do, s in zip(d_out, subs)]
    got = P.assemble(case, maps, parts)
    for a, b in zip(got, got_whole):
        assert np.array_equal(a, b)
    c = round_case_to_f32(case) if prec == "f32" else case
    err, _ = field_errors(got, oracle_rhs(c), joint_momentum=prec == "f32")
    assert err.max() < (1e-11 if prec == "f64" else 2e-4), err
    # one RK45[2R+] step on the internal states
    for cx, s in zip(ctxs, subs):
        cx.set_state(s["u0"])
    for i in range(5):
        for ph in range(3):
            for cx in ctxs:
                cx.rk_stage_phase(dt, i, ph)
            torch.cuda.synchronize()
            if ph < 2:
                H.local_exchange(xchs, ph)
                torch.cuda.synchronize()
    st = P.assemble(case, maps, [cx.get_state() for cx in ctxs])
    for a, b in zip(st, st_whole):
        assert np.array_equal(a, b)
    for cx in ctxs:
        cx.close()
