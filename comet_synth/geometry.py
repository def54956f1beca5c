"""Stand-in cylindrical drift chamber (BASELINE.json configs[0]; reading R18).

20 sense layers at r_i = 53.0 + 1.6 i cm, n_i = 198 + 6 i wires per layer,
wire endpoints at z = -/+ 75 cm.  Wire k of layer i has its z = -75 endpoint at
azimuth 2 pi k / n_i and its z = +75 endpoint at 2 pi k / n_i + s_i * 0.07 rad
with s_i = +1 for even i and -1 for odd i (the alternating stereo of
PAPER.md:47).  Both endpoints sit at radius r_i.  5100 wires in total.
"""
from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class CDCGeometry:
    wire_a: np.ndarray      # [3][n_wires] float64, endpoint at z = -half_len
    wire_b: np.ndarray      # [3][n_wires] float64, endpoint at z = +half_len
    layer: np.ndarray       # [n_wires] int32
    layer_radius: np.ndarray  # [n_layers] float64
    half_len: float

    @property
    def n_wires(self) -> int:
        return int(self.wire_a.shape[1])

    @property
    def n_layers(self) -> int:
        return int(self.layer_radius.shape[0])


def cdc_geometry(n_layers: int = 20, r0: float = 53.0, dr: float = 1.6,
                 n0: int = 198, dn: int = 6, half_len: float = 75.0,
                 stereo: float = 0.07) -> CDCGeometry:
    a_cols, b_cols, lay = [], [], []
    radii = np.empty(n_layers)
    for i in range(n_layers):
        r = r0 + dr * i
        n = n0 + dn * i
        radii[i] = r
        az = 2.0 * np.pi * np.arange(n) / n
        s = 1.0 if i % 2 == 0 else -1.0
        az_b = az + s * stereo
        a_cols.append(np.stack([r * np.cos(az), r * np.sin(az), np.full(n, -half_len)]))
        b_cols.append(np.stack([r * np.cos(az_b), r * np.sin(az_b), np.full(n, +half_len)]))
        lay.append(np.full(n, i, dtype=np.int32))
    return CDCGeometry(
        wire_a=np.ascontiguousarray(np.concatenate(a_cols, axis=1)),
        wire_b=np.ascontiguousarray(np.concatenate(b_cols, axis=1)),
        layer=np.concatenate(lay),
        layer_radius=radii,
        half_len=half_len,
    )
