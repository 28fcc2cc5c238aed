"""Shared plumbing of the -m gpu parity tests: move seeded inputs to the device, run the
CUDA path through the C-ABI binding, bring canonical results back.  No operator arithmetic."""
import numpy as np
import torch

import paper_2211_13719_b200 as mrhs

TOL = 1e-5   # BASELINE.json north_star: relative L2 per RHS, fp32 path vs fp64 oracle (reading S16)


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def host(t):
    return t.detach().cpu().numpy()


def make_wilson(dims, nrhs, mass, csw, U, clover=None):
    return mrhs.Wilson(dims, nrhs, mass, csw, dev(U), None if clover is None else dev(clover))


def gpu_dhop(w, psi):
    d_in = w.import_field(dev(psi), mrhs.FULL)
    d_out = w.empty(mrhs.FULL)
    w.dhop(d_in, d_out)
    torch.cuda.synchronize()
    return host(w.export_field(d_out, mrhs.FULL))


def gpu_meooe(w, psi_cb, out_parity):
    d_in = w.import_field(dev(psi_cb), 1 - out_parity)
    d_out = w.empty(out_parity)
    w.meooe(d_in, d_out, out_parity)
    torch.cuda.synchronize()
    return host(w.export_field(d_out, out_parity))


def gpu_mooee(w, psi, parity):
    d_in = w.import_field(dev(psi), parity)
    d_out = w.empty(parity)
    w.mooee(d_in, d_out, parity)
    torch.cuda.synchronize()
    return host(w.export_field(d_out, parity))
