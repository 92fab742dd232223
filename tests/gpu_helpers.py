"""Run the CUDA path through the C-ABI binding on workload inputs (GPU tests only)."""
import numpy as np
import torch

from paper_1706_08563_b200 import prism

DEV = torch.device("cuda:0")


def ws(p, which, n_atoms=0):
    return torch.empty(prism.workspace_bytes(p, which, n_atoms), dtype=torch.uint8, device=DEV)


def gpu_potential(w, p=None, phonon=0, on_host=False):
    p = p or prism.params_from_workload(w)
    p.potential_on_host = 1 if on_host else 0
    lut_z, r_cut, lut_v = w.lut()
    shape = (w.n_slices, w.ny, w.nx)
    v = (torch.empty(shape, dtype=torch.float32).pin_memory() if on_host
         else torch.empty(shape, dtype=torch.float32, device=DEV))
    prism.build_potential(p, w.atoms_for_phonon(phonon), w.z, lut_z, r_cut, lut_v, v,
                          ws(p, prism.WS_POTENTIAL, len(w.z)))
    torch.cuda.synchronize()
    return v


def gpu_smatrix(w, v, p=None):
    p = p or prism.params_from_workload(w)
    p.potential_on_host = 0 if v.is_cuda else 1
    s = torch.empty((prism.num_beams(p), w.ny, w.nx), dtype=torch.complex64, device=DEV)
    beams = prism.compute_smatrix(p, v, s, ws(p, prism.WS_SMATRIX))
    torch.cuda.synchronize()
    return s, beams


def gpu_prism_output(w, s, beams, p=None, host_out=False):
    p = p or prism.params_from_workload(w)
    shape = (w.probes_y, w.probes_x, prism.num_bins(p))
    out = (torch.empty(shape, dtype=torch.float32).pin_memory() if host_out
           else torch.empty(shape, dtype=torch.float32, device=DEV))
    prism.compute_output(p, s, beams, out, ws(p, prism.WS_OUTPUT))
    torch.cuda.synchronize()
    return out.cpu().numpy().astype(np.float64).reshape(-1, shape[-1])


def gpu_multislice(w, v, p=None, host_out=False):
    p = p or prism.params_from_workload(w)
    p.potential_on_host = 0 if v.is_cuda else 1
    shape = (w.probes_y, w.probes_x, prism.num_bins(p))
    out = (torch.empty(shape, dtype=torch.float32).pin_memory() if host_out
           else torch.empty(shape, dtype=torch.float32, device=DEV))
    prism.multislice_output(p, v, out, ws(p, prism.WS_MULTISLICE))
    torch.cuda.synchronize()
    return out.cpu().numpy().astype(np.float64).reshape(-1, shape[-1])


def dark_field(w, p):
    """Index of the first ring entirely beyond the probe semi-angle."""
    return int(np.ceil(w.alpha / w.det_step)) + 1
