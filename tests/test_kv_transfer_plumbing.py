"""-m "not gpu": the two-worker KV transfer path (paper_2607_04206_b200/kv_transfer.py) with
world size 2 on gloo.  The kernels cannot run without a GPU, so gather / scatter are numpy stand-ins (the oracle's); what is
exercised is the N > 1 plumbing: header framing, per-layer ordering of the sends, page remapping on the receiver."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, os.environ["SANGAM_ROOT"])
import numpy as np, torch, torch.distributed as dist
from paper_2607_04206_b200 import kv_transfer as kt
from oracle import neighbours as nb
rank = int(os.environ["RANK"])
dist.init_process_group(backend="gloo")
P, Hkv, D, LAYERS = 40, 2, 8, 3
g = np.random.default_rng(77)                        # both ranks draw the same reference content
pools = [(g.integers(0, 65535, (P, Hkv, 16, D)).astype(np.int16), g.integers(0, 65535, (P, Hkv, 16, D)).astype(np.int16)) for _ in range(LAYERS)]
src_ids = np.array([5, 17, 3, 30, 8], np.int32); dst_ids = np.array([0, 1, 2, 9, 4], np.int32)
new_stage = lambda n: (torch.zeros((n, Hkv, 16, D), dtype=torch.int16), torch.zeros((n, Hkv, 16, D), dtype=torch.int16))
def gather(kp, vp, ids, ks, vs):
    a, b = nb.kv_gather(kp.numpy(), vp.numpy(), ids.numpy()); ks.copy_(torch.from_numpy(a)); vs.copy_(torch.from_numpy(b))
def scatter(ks, vs, ids, kp, vp):
    nb.kv_scatter(ks.numpy(), vs.numpy(), ids.numpy(), kp.numpy(), vp.numpy())
if rank == 0:
    layers = [(torch.from_numpy(k.copy()), torch.from_numpy(v.copy())) for k, v in pools]
    kt.send_request_kv(dist, 1, req_id=4242, ctx_len=77, page_ids=torch.from_numpy(src_ids), layers=layers, gather=gather, new_stage=new_stage)
    print(json.dumps({"rank": 0, "ok": True}))
else:
    layers = [(torch.zeros((P, Hkv, 16, D), dtype=torch.int16), torch.zeros((P, Hkv, 16, D), dtype=torch.int16)) for _ in range(LAYERS)]
    rid, c, ids = kt.recv_request_kv(dist, 0, layers, alloc_pages=lambda n: torch.from_numpy(dst_ids[:n].copy()), scatter=scatter, new_stage=new_stage, device="cpu")
    ok = rid == 4242 and c == 77 and ids.tolist() == dst_ids.tolist()
    for (kd, vd), (ks, vs) in zip(layers, pools):
        for s, t in zip(src_ids, dst_ids):
            ok = ok and np.array_equal(kd.numpy()[t], ks[s]) and np.array_equal(vd.numpy()[t], vs[s])
        rest = [p for p in range(P) if p not in dst_ids.tolist()]
        ok = ok and not kd.numpy()[rest].any() and not vd.numpy()[rest].any()
    print(json.dumps({"rank": 1, "ok": bool(ok)}))
dist.barrier()
dist.destroy_process_group()
"""


def test_request_kv_transfer_world2_gloo():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    procs = []
    for r in range(2):
        e = dict(os.environ)
        e.update({"RANK": str(r), "LOCAL_RANK": str(r), "WORLD_SIZE": "2", "MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port),
                  "SANGAM_ROOT": ROOT, "CUDA_VISIBLE_DEVICES": ""})
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER], env=e, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=180) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e[-2000:]
    vals = [json.loads(o.strip().splitlines()[-1]) for o, _ in outs]
    assert all(v["ok"] for v in vals)
