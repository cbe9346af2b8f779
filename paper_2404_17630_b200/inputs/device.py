"""Device-side builds of the big workloads (configs 3 and 4 at full size): the same recipes as
inputs/configs.py with torch doing the array plumbing on the GPU (hash RNG in int64 two's
complement, cuFFT for the Gaussian field, meshgen's device kernels for the Voronoi mesh), so a
384^3 mesh (~30 GB of geometry) never touches the host.  Input generation only.
"""
import numpy as np

from . import configs as cfg
from . import mesh as M


def _s64(x):
    x &= (1 << 64) - 1
    return x - (1 << 64) if x >= (1 << 63) else x


_M1, _M2, _M3, _MS = (_s64(v) for v in (0x9E3779B97F4A7C15, 0xBF58476D1CE4E5B9, 0x94D049BB133111EB, 0x632BE59BD9B4E019))


def _lsr(z, k):
    return (z >> k) & ((1 << (64 - k)) - 1)


def mix(z):
    z = z + _M1
    z = (z ^ _lsr(z, 30)) * _M2
    z = (z ^ _lsr(z, 27)) * _M3
    return z ^ _lsr(z, 31)


def u01(seed, stream, index):
    """Same bits as inputs.rng.u01; index: int64 tensor."""
    import torch
    base = mix(torch.tensor(_s64(int(seed) + int(stream) * 0x632BE59BD9B4E019), dtype=torch.int64, device=index.device))
    z = mix(base ^ index)
    return _lsr(z, 11).to(torch.float64) * (2.0 ** -53)


def normal(seed, stream, index):
    import torch
    u1 = u01(seed, 2 * stream, index)
    u2 = u01(seed, 2 * stream + 1, index)
    return torch.sqrt(-2.0 * torch.log(1.0 - u1)) * torch.cos(2.0 * np.pi * u2)


def gaussian_field(n, seed, dev):
    import torch
    idx = torch.arange(n ** 3, dtype=torch.int64, device=dev)
    w = normal(seed, 0, idx).reshape(n, n, n)
    del idx
    k = torch.fft.fftfreq(n, device=dev, dtype=torch.float64) * n
    k2 = k[:, None, None] ** 2 + k[None, :, None] ** 2 + k[None, None, :] ** 2
    amp = torch.where(k2 > 0, 1.0 / torch.sqrt(torch.clamp(k2, min=1e-300)), torch.zeros_like(k2))
    del k2
    g = torch.fft.ifftn(torch.fft.fftn(w) * amp).real
    del w, amp
    return (g / g.std(unbiased=False)).reshape(-1)


def cfl_dt(mesh, ctilde, eta=0.3):
    import torch
    sa = torch.zeros(mesh.ncell, dtype=torch.float64, device=mesh.area.device)
    sa.index_add_(0, mesh.left.long(), mesh.area)
    ok = mesh.right >= 0
    sa.index_add_(0, mesh.right[ok].long(), mesh.area[ok])
    return float(eta * torch.min(6.0 * mesh.volume / sa).item() / ctilde)


def config34_device(n, c, device="cuda:0"):
    """Reionisation-like periodic volume built on the device.  Returns a cfg.Workload whose mesh and
    state arrays are cuda tensors (sources stay on the host: they are few)."""
    import torch
    dev = torch.device(device)
    full = 256 if c == 3 else 384
    nsrc_full = 10000 if c == 3 else 34000
    nsrc = max(1, int(round(nsrc_full * (n / full) ** 3)))
    g = gaussian_field(n, cfg.SEED_RHO + c, dev)
    nH = 2.0e-4 * torch.exp(1.5 * g - 0.5 * 1.5 ** 2)
    del g
    top = torch.topk(nH, nsrc).indices
    cells = torch.sort(top).values
    lg = 50.0 + 3.0 * u01(cfg.SEED_SRC + c, 0, cells)
    rate = (torch.as_tensor(cfg.SHARE3, device=dev)[:, None] * (10.0 ** lg)[None, :]).cpu().numpy()
    src = cfg.Sources(cells.to(torch.int32).cpu().numpy(), np.ascontiguousarray(rate))
    spacing = 10.0 * cfg.KPC
    mesh = M.voronoi_device(n, n * spacing, 0.3, cfg.SEED_MESH + c, True, device=device)
    ct = 0.2 * cfg.C_LIGHT
    p = cfg._hhe_params(ct)
    C = mesh.ncell
    z = lambda *s: torch.zeros(*s, dtype=torch.float64, device=dev)
    xHII = torch.full((C,), 1.0e-6, dtype=torch.float64, device=dev)
    xHeII = torch.full((C,), 1.0e-6, dtype=torch.float64, device=dev)
    xHeIII = z(C)
    xe = xHII + cfg.Y_HE * (xHeII + 2.0 * xHeIII)
    eth = 1.5 * nH * (1.0 + cfg.Y_HE + xe) * cfg.K_B * 1.0e4
    st = cfg.State(z(3, C), z(3, 3, C), xHII, xHeII, xHeIII, eth, nH)
    return cfg.Workload("config%d_reion_%d" % (c, n), mesh, p, st, src, cfl_dt(mesh, ct), {"spacing": spacing})
