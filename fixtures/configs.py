"""The five BASELINE.json configs (plus small test variants) as plain records.

BASELINE.json:configs[0..4]; SURVEY.md section 8(d) and Appendix C.
sym: 0 = U(1)xU(1) (twoS is 2*Sz), 1 = SU(2) (twoS is 2*S).
`bond` = number of orbitals in the left block; the two-site window is sites
(bond, bond+1); the right block holds sites bond+2 .. L-1.
"""
from dataclasses import dataclass, replace

SYM_U1U1 = 0
SYM_SU2 = 1


@dataclass(frozen=True)
class Config:
    name: str
    L: int
    N: int
    twoS: int
    sym: int
    D: int
    n_chol: int
    bond: int
    hdiag: str = "default"   # "default" | "spread" | "bands"
    sigma_N: float = 2.0
    sigma_Z: float = 1.5     # abelian spread of (n_up - n_dn)
    sigma_S: float = 2.0     # SU(2) spread of S

    def with_(self, **kw):
        return replace(self, **kw)


CONFIGS = {
    "cfg0": Config("cfg0", L=8, N=8, twoS=0, sym=SYM_U1U1, D=256, n_chol=16, bond=3),
    "cfg1": Config("cfg1", L=24, N=24, twoS=0, sym=SYM_U1U1, D=512, n_chol=32, bond=11),
    # cfg1 with a 4x larger block-state budget: same integrals and recipe, sector dimensions ~100-190
    # (the size class of configs[2]); bench.py --config cfg1_d2048 shows the kernels at that scale
    "cfg1_d2048": Config("cfg1_d2048", L=24, N=24, twoS=0, sym=SYM_U1U1, D=2048, n_chol=32, bond=11),
    "cfg2": Config("cfg2", L=36, N=54, twoS=0, sym=SYM_SU2, D=2048, n_chol=48, bond=17,
                   hdiag="spread"),
    "cfg3": Config("cfg3", L=36, N=54, twoS=0, sym=SYM_SU2, D=4096, n_chol=48, bond=17,
                   hdiag="spread"),
    "cfg4": Config("cfg4", L=102, N=89, twoS=5, sym=SYM_SU2, D=1024, n_chol=96, bond=50,
                   hdiag="bands"),
}


def get_config(name: str) -> Config:
    return CONFIGS[name]
