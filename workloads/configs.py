"""Workload table mirroring BASELINE.json:configs[0..4] (ids 1..5) plus small test-only shapes.

Fields: cell (orthorhombic edge lengths, bohr), kpoints (reduced), Ecut (Ha), S (FFT box), nb (bands
per k), natoms, n_lm (projectors per atom: 4 = s,p ; 9 = s,p,d), atoms (placement rule), extra
(additional term in V).  Exact nG per (config, k) is in tests/golden/basis_counts.txt.
"""

CONFIGS = {
    1: dict(name="cfg1_cubic10_G_32^3", cell=(10.0, 10.0, 10.0), kpoints=[(0.0, 0.0, 0.0)], Ecut=10.0,
            S=(32, 32, 32), nb=8, natoms=2, n_lm=4, atoms="uniform", extra="noise"),
    2: dict(name="cfg2_cubic20.5_k.25_80^3", cell=(20.5, 20.5, 20.5), kpoints=[(0.25, 0.25, 0.25)], Ecut=15.0,
            S=(80, 80, 80), nb=128, natoms=64, n_lm=4, atoms="uniform", extra=None),
    3: dict(name="cfg3_molbox30_G_128^3", cell=(30.0, 30.0, 30.0), kpoints=[(0.0, 0.0, 0.0)], Ecut=20.0,
            S=(128, 128, 128), nb=256, natoms=32, n_lm=9, atoms="clustered", extra="cavity"),
    4: dict(name="cfg4_slab20x20x60_4k_72x72x216", cell=(20.0, 20.0, 60.0),
            kpoints=[(0.0, 0.0, 0.0), (0.5, 0.0, 0.0), (0.0, 0.5, 0.0), (0.5, 0.5, 0.0)], Ecut=15.0,
            S=(72, 72, 216), nb=384, natoms=96, n_lm=4, atoms="slab", extra="ramp"),
    5: dict(name="cfg5_bulk216_G_128^3", cell=(30.7, 30.7, 30.7), kpoints=[(0.0, 0.0, 0.0)], Ecut=20.0,
            S=(128, 128, 128), nb=512, natoms=216, n_lm=4, atoms="lattice6", extra=None),
}

# Small shapes for parity tests: every radix (2, 3, 5) and mixed lengths, non-cubic boxes, k != 0,
# sizes that span several tiles of the CUDA kernels and leave ragged tails.
TEST_CONFIGS = {
    101: dict(name="t_12x15x20", cell=(6.0, 7.5, 9.0), kpoints=[(0.1, -0.2, 0.3)], Ecut=4.0,
              S=(12, 15, 20), nb=5, natoms=2, n_lm=4, atoms="uniform", extra="noise"),
    102: dict(name="t_30x36x40", cell=(9.0, 11.0, 12.5), kpoints=[(0.25, 0.0, -0.4)], Ecut=8.0,
              S=(30, 36, 40), nb=19, natoms=5, n_lm=9, atoms="uniform", extra="noise"),
    103: dict(name="t_48x45x50", cell=(14.0, 13.0, 15.0), kpoints=[(0.0, 0.0, 0.0), (0.5, 0.5, 0.5)], Ecut=9.0,
              S=(48, 45, 50), nb=37, natoms=11, n_lm=4, atoms="uniform", extra="ramp"),
    104: dict(name="t_64^3", cell=(16.0, 16.0, 16.0), kpoints=[(0.0, 0.0, 0.0)], Ecut=12.0,
              S=(64, 64, 64), nb=33, natoms=17, n_lm=4, atoms="lattice6", extra=None),
    105: dict(name="t_27x25x32", cell=(8.0, 7.0, 9.5), kpoints=[(0.3, 0.3, 0.1)], Ecut=7.0,
              S=(27, 25, 32), nb=9, natoms=3, n_lm=9, atoms="clustered", extra="cavity"),
}


# Boxes that put every additional specialised FFT length (48 96 100 120 144 160 192 256) on every axis (each axis runs
# different kernels: columns = axis 2, rows = axis 1, planes = axis 0); cell edge = S/4 bohr, Ecut 9 Ha => |m_d| <~ S_d/6.
def _rot(name, S, cfg_id):
    return dict(name=name, cell=tuple(s / 4.0 for s in S), kpoints=[(0.0, 0.0, 0.0) if cfg_id % 2 else (0.3, -0.2, 0.1)],
                Ecut=9.0, S=S, nb=3, natoms=2, n_lm=4, atoms="uniform", extra="noise")


_LEN_BOXES = [(48, 96, 100), (96, 100, 48), (100, 48, 96), (120, 144, 160), (144, 160, 120), (160, 120, 144),
              (192, 256, 32), (256, 32, 192), (32, 192, 256)]
TEST_CONFIGS[210] = _rot("t_len_72x40x48", (72, 40, 48), 210)   # plane length 72: the two-pencils-per-thread K3
TEST_CONFIGS[216] = _rot("t_len_24x32x128", (24, 32, 128), 216)  # column length 128: two-round first pass in K1
TEST_CONFIGS[214] = _rot("t_len_128x80x27", (128, 80, 27), 214)  # odd S2: the pair / hybrid kernels must step aside
TEST_CONFIGS[215] = _rot("t_len_72x128x25", (72, 128, 25), 215)
TEST_CONFIGS[213] = _rot("t_len_24x128x32", (24, 128, 32), 213)  # row length 128: hybrid pair/single K2, K4
TEST_CONFIGS[212] = _rot("t_len_128x24x32", (128, 24, 32), 212)  # plane length 128: hybrid pair/single K3
TEST_CONFIGS[211] = _rot("t_len_80x27x32", (80, 27, 32), 211)   # plane length 80: two tiles per CTA, odd S1 (idle group)
# plane length 80 with |m0| up to 22 >= 2 R2 = 20: K3's pruned radix-8 butterflies must step aside
TEST_CONFIGS[217] = dict(_rot("t_len_80x27x32_wide", (80, 27, 32), 217), Ecut=25.0)
for _i, _S in enumerate(_LEN_BOXES):
    TEST_CONFIGS[201 + _i] = _rot("t_len_%dx%dx%d" % _S, _S, 201 + _i)


def get_config(cfg_id):
    if cfg_id in CONFIGS:
        return CONFIGS[cfg_id]
    return TEST_CONFIGS[cfg_id]
