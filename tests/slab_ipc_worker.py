"""Worker of test_slabs_gpu.py::test_two_processes_cuda_ipc / test_two_ranks_two_gpus_nccl -- launched by
torch.distributed.run with two ranks: each rank owns one z-slab (slabs.RankSlab), rank 0 gathers the
result and writes it to the .npz given as argv[1].  argv[3] = "gloo" (default: both ranks on GPU 0, host
barrier per step) or "nccl" (rank r on GPU r: peer stores over NVLink, one-element all-reduce per step)."""
import sys

import numpy as np

STEPS = 8


def case(jet):
    from paper_2403_15773_b200 import inputs
    nx, ny, nz = 64, 16, 21
    if jet:
        prm = inputs.jet_params(nx, ny, nz, D=7, U=0.04, Re=300.0, We=50.0, perturbation=0.1, seed=11)
        d = inputs.jet_developed(nx, ny, nz, D=7, ndrop=3)
    else:
        prm = dict(nx=nx, ny=ny, nz=nz, omega=1.8, two_component=True, sigma=0.01, interface_width=3.0)
        d = inputs.smooth_random(nx, ny, nz, seed=13)
    d = {k: (None if v is None else np.asarray(v, dtype=np.float32)) for k, v in d.items()}
    return d, prm


def main():
    import torch.distributed as dist
    from paper_2403_15773_b200 import slabs, tslb
    import os
    import torch
    out, jet = sys.argv[1], sys.argv[2] == "1"
    backend = sys.argv[3] if len(sys.argv) > 3 else "gloo"
    device = int(os.environ.get("LOCAL_RANK", "0")) if backend == "nccl" else 0
    torch.cuda.set_device(device)
    if backend == "nccl":
        dist.init_process_group("nccl", device_id=torch.device("cuda", device))
    else:
        dist.init_process_group("gloo")
    d, prm = case(jet)
    kw = {k: v for k, v in prm.items() if k not in ("nx", "ny", "nz", "omega")}
    s = slabs.RankSlab(prm["nx"], prm["ny"], prm["nz"], prm["omega"], precision=tslb.F32, device=device, **kw)
    z0, z1 = s.z0, s.z1
    pq = None if d.get("pineq") is None else [np.ascontiguousarray(a[z0:z1]) for a in d["pineq"]]
    s.init_fields(*[np.ascontiguousarray(d[k][z0:z1]) for k in ("rho", "ux", "uy", "uz")],
                  np.ascontiguousarray(d["phi"][z0:z1]), pq)
    s.step(STEPS)
    m = s.get_moments()
    parts = [None] * dist.get_world_size()
    dist.all_gather_object(parts, m)
    if dist.get_rank() == 0:
        full = {k: np.concatenate([p[k] for p in parts], axis=1 if k == "pineq" else 0) for k in m}
        np.savez(out, **full)
    s.close()
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
