"""Helpers for the `-m gpu` parity tests: seeded pools on the device (torch = memory + streams only),
mirrored on the host for the oracle.  Holds none of the method's arithmetic."""
from __future__ import annotations

import numpy as np
import torch

import paper_2406_03243_b200 as llx
import synth

SENT = synth.SENTINEL_U16


def tile_elems(g):
    return g["block_size"] * g["kv_heads"] * g["head_dim"]


class DevPool:
    """A torch-owned device buffer wrapped as an llx pool, viewed as int16 [L,2,num_blocks,tile_elems]."""

    def __init__(self, g, num_blocks=None, fill=None, dtype=llx.F16):
        self.g = dict(g)
        self.nb = int(num_blocks if num_blocks is not None else g["num_blocks"])
        self.te = tile_elems(g)
        nbytes = llx.pool_bytes_for(g["layers"], g["kv_heads"], g["head_dim"], g["block_size"], dtype, self.nb)
        self.raw = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        self.view = self.raw.view(torch.int16).view(g["layers"], 2, self.nb, self.te)
        if fill is not None:
            self.view.fill_(int(np.array(fill, dtype=np.uint16).view(np.int16)))
        self.pool = llx.pool_wrap(self.raw.data_ptr(), nbytes, g["layers"], g["kv_heads"], g["head_dim"],
                                  g["block_size"], dtype, self.nb, keepalive=self.raw)

    def upload_slice(self, layer, kv, arr_u16: np.ndarray):
        self.view[layer, kv].copy_(torch.from_numpy(np.ascontiguousarray(arr_u16).view(np.int16)))

    def fill_from_synth(self, seed, pool_id, layers=None):
        for l in (range(self.g["layers"]) if layers is None else layers):
            for kv in range(2):
                self.upload_slice(l, kv, synth.slice_values_f16(seed, pool_id, l, kv, self.nb, self.te))

    def fill_device_random(self, seed):
        """Seeded device-side fill (input generation only) for layers the host does not mirror."""
        gen = torch.Generator(device="cuda")
        gen.manual_seed(seed)
        flat = self.raw.view(torch.int16)
        step = 1 << 28
        for a in range(0, flat.numel(), step):
            b = min(flat.numel(), a + step)
            # arbitrary 16-bit patterns: migration is a bit copy and never interprets them
            flat[a:b] = torch.randint(-0x3C00, 0x3C00, (b - a,), generator=gen, device="cuda", dtype=torch.int16)

    def host(self) -> np.ndarray:
        torch.cuda.synchronize()
        return self.view.cpu().numpy().view(np.uint16)

    def host_layer(self, layer) -> np.ndarray:
        torch.cuda.synchronize()
        return self.view[layer:layer + 1].cpu().numpy().view(np.uint16)


def host_pool_from_synth(g, seed, pool_id, num_blocks=None, layers=None):
    nb = int(num_blocks if num_blocks is not None else g["num_blocks"])
    te = tile_elems(g)
    ls = list(range(g["layers"])) if layers is None else list(layers)
    out = np.empty((len(ls), 2, nb, te), dtype=np.uint16)
    for j, l in enumerate(ls):
        for kv in range(2):
            out[j, kv] = synth.slice_values_f16(seed, pool_id, l, kv, nb, te)
    return out


def first_mismatch(got: np.ndarray, want: np.ndarray) -> str:
    """(layer, kv, block, element, expected, got) of the first differing word."""
    idx = np.argwhere(got != want)
    if idx.size == 0:
        return "equal"
    l, kv, b, e = idx[0]
    return (f"{idx.shape[0]} words differ; first at layer={l} kv={kv} block={b} elem={e}: "
            f"expected 0x{int(want[l, kv, b, e]):04x} got 0x{int(got[l, kv, b, e]):04x}")


def assert_pool_equal(got: np.ndarray, want: np.ndarray):
    assert got.shape == want.shape
    assert np.array_equal(got, want), first_mismatch(got, want)
