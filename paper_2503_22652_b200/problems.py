"""Upload a seeded workload (a dict from the `workloads` package: inputs only, no method
arithmetic) to the GPU as the operator specs `Rchfsi` takes."""


def upload_problem(prob, device="cuda:0", fe_cells_f32_only=False):
    """Returns (A_spec, B_spec or None, dinv tensor or None)."""
    import numpy as np
    import torch
    dev = torch.device(device)

    def t(a, dtype):
        return torch.as_tensor(np.ascontiguousarray(a), dtype=dtype).to(dev)

    kind = prob["kind"]
    B = None
    if kind == "dense":
        A = dict(kind="dense", A=t(prob["A"], torch.float64))
        if prob.get("B") is not None:
            B = dict(kind="dense", A=t(prob["B"], torch.float64))
    elif kind == "csr":
        A = dict(kind="csr", rowptr=t(prob["rowptr"], torch.int64), colind=t(prob["colind"], torch.int32),
                 vals=t(prob["vals"], torch.float64))
    elif kind == "fe":
        conn = t(prob["conn"], torch.int32)
        if fe_cells_f32_only or prob["A_cells"].dtype == np.float32:
            A = dict(kind="fe", conn=conn, m=prob["m"], cell_mats_f32=t(prob["A_cells"], torch.float32))
        else:
            A = dict(kind="fe", conn=conn, m=prob["m"], cell_mats=t(prob["A_cells"], torch.float64))
        B = dict(kind="fe", conn=conn, m=prob["m"], cell_mats=t(prob["B_cell"], torch.float64), shared=True)
    else:
        raise ValueError(kind)
    dinv = t(prob["dinv"], torch.float64) if prob.get("dinv") is not None else None
    return A, B, dinv
