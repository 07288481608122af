"""Architecture descriptions (plain data) for the configs of BASELINE.json.

PAPER.md L262 (App. B): k = 16, EdgeConv channels (64,64,64),(128,128,128),(256,256,256), FC 256 -> 2,
two coordinates.  The number of input features follows BASELINE.json configs (reading R1).
"""
from dataclasses import dataclass, field
from typing import List, Tuple


@dataclass(frozen=True)
class Arch:
    in_features: int
    k: int
    channels: Tuple[Tuple[int, int, int], ...]
    fc_hidden: Tuple[int, ...]
    n_classes: int = 2
    coord_dims: int = 2
    max_particles: int = 128

    @property
    def n_blocks(self) -> int:
        return len(self.channels)

    def block_in(self, l: int) -> int:
        return self.in_features if l == 0 else self.channels[l - 1][2]

    def with_features(self, f: int) -> "Arch":
        return Arch(f, self.k, self.channels, self.fc_hidden, self.n_classes, self.coord_dims, self.max_particles)


def weight_count(a: Arch) -> int:
    """Number of fp32 values in the flat blob (layout: include/gnn.h, "Weight blob")."""
    n = 0
    for l, (c1, c2, c3) in enumerate(a.channels):
        cin = a.block_in(l)
        for (i, o) in ((2 * cin, c1), (c1, c2), (c2, c3)):
            n += o * i + 2 * o
        n += c3 * cin + 2 * c3
    i = a.channels[-1][2]
    for d in tuple(a.fc_hidden) + (a.n_classes,):
        n += d * i + d
        i = d
    return n


ARCHS = {
    # BASELINE.json configs[0]
    "tiny": Arch(in_features=4, k=4, channels=((32, 32, 32),), fc_hidden=(), max_particles=16),
    # configs[1], [3]; PAPER.md L262 shape with F = 7
    "particlenet": Arch(in_features=7, k=16, channels=((64, 64, 64), (128, 128, 128), (256, 256, 256)),
                        fc_hidden=(256,), max_particles=128),
    # configs[2]: F = 9
    "particlenet_f9": Arch(in_features=9, k=16, channels=((64, 64, 64), (128, 128, 128), (256, 256, 256)),
                           fc_hidden=(256,), max_particles=128),
    # configs[4] wide variant
    "wide": Arch(in_features=7, k=16, channels=((128, 128, 128), (256, 256, 256), (512, 512, 512)),
                 fc_hidden=(512,), max_particles=128),
    # PAPER.md L262 literal: five input features
    "paper_f5": Arch(in_features=5, k=16, channels=((64, 64, 64), (128, 128, 128), (256, 256, 256)),
                     fc_hidden=(256,), max_particles=128),
}
