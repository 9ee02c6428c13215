"""B200-native single-pulse-search hot path behind AMBER's auto-tuning (arXiv:1811.04165).

The product is the C-ABI library `libddp.so` (include/ddp.h; sources in csrc/): brute-force
incoherent dedispersion (direct and two-step subband), decimating boxcar integration, per-(DM,
width) S/N, and the GA / brute-force / random tuners that time those kernels.  This package is the
thin Python binding (same names as the C entry points, argument marshalling only) plus a helper
that allocates the device buffers of a plan with PyTorch.
"""
from __future__ import annotations

from .binding import (DDP_NSLOTS, K_DIRECT, K_INTEGRATE, K_ISNR, K_SNR, K_SUB1, K_SUB2, KCACHE_DIR, KERNEL_NAMES,
                      STAGE_DIRECT, STAGE_SMEM, STAGE_TMA, SYMBOLS, DdpError, Kcfg, Plan, PlanInfo, TuneIo,
                      lib, make_tune_io, plan_create, status_str, version)

__all__ = ["plan_create", "Plan", "Kcfg", "PlanInfo", "TuneIo", "DdpError", "make_tune_io", "alloc_buffers",
           "plan_from_config", "lib", "status_str", "version", "SYMBOLS", "KERNEL_NAMES", "DDP_NSLOTS",
           "K_DIRECT", "K_SUB1", "K_SUB2", "K_INTEGRATE", "K_SNR", "K_ISNR", "STAGE_DIRECT", "STAGE_SMEM", "STAGE_TMA",
           "KCACHE_DIR"]


def plan_from_config(cfg, **kw) -> Plan:
    """Plan of a `synth.configs.SearchConfig`-shaped object (pure data: frequencies, DM grid, widths)."""
    sb = getattr(cfg, "subband", None)
    if sb is not None:
        return plan_create(cfg.chan_freq_mhz(), cfg.t_samp_s, None, cfg.widths, cfg.nsamp_out,
                           n_subbands=sb.n_subbands, n_coarse=sb.n_coarse, coarse_dm_first=sb.coarse_first,
                           coarse_dm_step=sb.coarse_step, n_fine=sb.n_fine, fine_dm_step=sb.fine_step, **kw)
    return plan_create(cfg.chan_freq_mhz(), cfg.t_samp_s, cfg.dm_list(), cfg.widths, cfg.nsamp_out, **kw)


def alloc_buffers(plan: Plan, device="cuda:0", bind: bool = True) -> dict:
    """Device buffers of one search, allocated with PyTorch (the library never allocates):
    d_in uint8 (int16-typed uint16 for a 16-bit plan) [nchan][in_stride], d_out int32-typed uint32 [ndm][out_stride], d_integ [integ_elems],
    d_snr float32 [ndm][nwidths], d_argmax [ndm][nwidths], workspace (delay tables + subband buffer)."""
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_1811_04165_b200 needs a CUDA device: there is no CPU fallback")
    i = plan.query()
    dev = torch.device(device)
    b = {
        "d_in": torch.zeros((i.nchan, i.in_stride_min), dtype=torch.uint8 if i.input_bits == 8 else torch.int16, device=dev),
        "d_out": torch.zeros((i.ndm, i.out_stride_min), dtype=torch.int32, device=dev),
        "d_integ": torch.zeros((max(1, i.integ_elems),), dtype=torch.int32, device=dev),
        "d_snr": torch.zeros((i.ndm, i.nwidths), dtype=torch.float32, device=dev),
        "d_argmax": torch.zeros((i.ndm, i.nwidths), dtype=torch.int32, device=dev),
        "workspace": torch.zeros((i.workspace_bytes,), dtype=torch.uint8, device=dev),
    }
    if bind:
        plan.bind_workspace(b["workspace"])
    return b
