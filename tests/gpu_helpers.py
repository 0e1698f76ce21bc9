"""Helpers for the -m gpu parity tests: move oracle-made buffers to the device and results back."""
from __future__ import annotations
import numpy as np
import torch
import paper_2607_04749_b200 as E


def upload(bufs: dict) -> dict:
    """{(dev, kind): numpy uint16/uint32} -> {(dev, kind): uint8 CUDA tensor} (empty buffers dropped)."""
    out = {}
    for key, a in bufs.items():
        if a.shape[0]:
            out[key] = torch.from_numpy(a.view(np.uint8).copy()).cuda()
    return out


def download(t: torch.Tensor, elem_bytes: int) -> np.ndarray:
    a = t.cpu().numpy()
    return a.view(np.uint16 if elem_bytes == 2 else np.uint32)


def run_gpu_migration(w_model, old_cfg, new_cfg, src_np: dict, device_map=None, flags=E.ETC_LOCAL_DIRECT,
                      sketch_method=E.ETC_SKETCH_AUTO, poison=0xA5):
    """Whole CUDA path.  Returns dict(overlap, need, hold, device_map, local_bytes, plan, dst {(n,k): np array})."""
    old, new = E.etc_layout_create(w_model, old_cfg), E.etc_layout_create(w_model, new_cfg)
    ov, need, hold = E.etc_cost_matrix(old, new)
    if device_map is None:
        dm, lb = E.etc_sketch(ov, method=sketch_method)
    else:
        dm = torch.tensor(np.asarray(device_map, np.int32)).cuda()
        lb = None
    plan = E.etc_plan_create(old, new, dm, flags)
    assert plan.validate() == 0                    # every work item inside its buffers (device-side bounds check)
    src = upload(src_np) if src_np is not None else None
    dst = E.alloc_buffers(new, fill=poison)
    staging = torch.full((max(plan.stats.staging_bytes, 16),), poison, dtype=torch.uint8, device="cuda")
    if src is not None:
        E.etc_migrate(plan, src, dst, staging)
    torch.cuda.synchronize()
    out_np = {}
    for n in range(new.n_dev):
        for k in new.kinds():
            eb = 4 if k else w_model["param_bytes"]
            if (n, k) in dst:
                out_np[(n, k)] = download(dst[(n, k)], eb)
            else:
                out_np[(n, k)] = np.zeros(0, np.uint16 if eb == 2 else np.uint32)
    return dict(old=old, new=new, overlap=ov.cpu().numpy(), need=need.cpu().numpy(), hold=hold.cpu().numpy(),
                device_map=dm.cpu().numpy(), local_bytes=None if lb is None else int(lb.item()), plan=plan, dst=out_np)
