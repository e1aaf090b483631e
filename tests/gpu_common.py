"""Helpers for the -m gpu parity tests: move a workload to the device, run the oracle on the same fp32 inputs."""
import numpy as np
import torch

import oracle
from paper_2507_21684_b200.binding import Sph


class Dev:
    def __init__(self, wl):
        dev = "cuda:0"
        self.x = torch.from_numpy(wl.x).to(dev)
        self.v = torch.from_numpy(wl.v).to(dev)
        self.rho = torch.from_numpy(wl.rho).to(dev)
        self.m = torch.from_numpy(wl.m).to(dev)
        self.h = torch.from_numpy(wl.h).to(dev)
        self.kind = torch.from_numpy(wl.kind).to(dev)


def build(wl, scale=1.0, sph=None, dev=None):
    sph = sph or Sph(0)
    dev = dev or Dev(wl)
    sph.build_cells(wl.domain, dev.x, dev.h)
    nnz = sph.neighbors(scale)
    return sph, dev, nnz


def oracle_lists(wl, scale=1.0, method=1):
    return oracle.neighbors(wl.domain, wl.x, wl.h, search_scale=scale, method=method)
