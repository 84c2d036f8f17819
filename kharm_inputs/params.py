"""Parameter sets of BASELINE.json's five configs, as plain dicts.

Keys are the fields of the C structs `kh_params` (include/kharm.h) and `kho_params`
(oracle/kho.h); each binding turns the dict into its own struct.
"""
import math

NG = 3
PRIM_NAMES = ("rho", "u", "ut1", "ut2", "ut3", "B1", "B2", "B3")

MINKOWSKI, KS, FMKS = 0, 1, 2
BC_PERIODIC, BC_OUTFLOW, BC_POLAR, BC_FIXED = 0, 1, 2, 3
BC_BLOCK = 4            # ghost layers owned by a neighbouring block (libkharm only: kh_link_blocks / kh_step_blocks)
RECON_MC, RECON_WENO5 = 0, 1
INV_1DW, INV_KASTAUN = 0, 1
FRAME_FLUID, FRAME_DRIFT, FRAME_NORMAL = 0, 1, 2
B_FLUX_CT, B_FACE_CT = 0, 1
EMF_ARITHMETIC, EMF_UPWIND, EMF_CENTRED = 0, 1, 2

FLOOR_DEFAULTS = dict(rho_min=1e-6, u_min=1e-8, r_char=10.0, bsq_over_rho_max=100.0, bsq_over_u_max=1e4,
                      u_over_rho_max=100.0, gamma_max=50.0, dt_growth_max=1.3)


def base_params(**kw):
    p = dict(coords=MINKOWSKI, a=0.0, hslope=0.3, poly_xt=0.82, poly_alpha=14.0, mks_smooth=0.5,
             n1=16, n2=16, n3=16, xmin=[0.0, 0.0, 0.0], xmax=[1.0, 1.0, 1.0], bc=[BC_PERIODIC] * 6,
             gamma=4.0 / 3.0, cfl=0.9, recon=RECON_MC, inverter=INV_1DW, fofc=0, floor_frame=FRAME_FLUID, transport=B_FLUX_CT, emf=EMF_ARITHMETIC)
    p.update(FLOOR_DEFAULTS)
    p.update(kw)
    return p


def r_horizon(a):
    return 1.0 + math.sqrt(1.0 - a * a)


def config_params(cfg, n=None, recon=None):
    """cfg in 1..5.  `n` overrides the resolution: int (cube / square) or (n1,n2,n3)."""
    def res(default):
        if n is None:
            return default
        if isinstance(n, int):
            return (n, n, n if default[2] > 1 else 1)
        return tuple(n)

    if cfg == 1:    # linear MHD mode, Minkowski, periodic unit cube, MC
        n1, n2, n3 = res((32, 32, 32))
        p = base_params(n1=n1, n2=n2, n3=n3, gamma=4.0 / 3.0, recon=RECON_MC)
    elif cfg == 2:  # magnetised Bondi, FMKS a=0, 128x128x1; outflow / fixed / polar / polar / periodic
        n1, n2, n3 = res((128, 128, 1))
        p = base_params(coords=FMKS, a=0.0, n1=n1, n2=n2, n3=n3, gamma=4.0 / 3.0, recon=RECON_MC,
                        xmin=[math.log(0.9 * 2.0), 0.0, 0.0], xmax=[math.log(50.0), 1.0, 2.0 * math.pi],
                        bc=[BC_OUTFLOW, BC_FIXED, BC_POLAR, BC_POLAR, BC_PERIODIC, BC_PERIODIC])
    elif cfg in (3, 4):  # FM torus, Kerr a=0.9375, FMKS; SANE 192x128x128 WENO5 / MAD 288x128x128 MC
        a = 0.9375
        n1, n2, n3 = res((192, 128, 128) if cfg == 3 else (288, 128, 128))
        p = base_params(coords=FMKS, a=a, n1=n1, n2=n2, n3=n3, gamma=13.0 / 9.0,
                        recon=RECON_WENO5 if cfg == 3 else RECON_MC,
                        xmin=[math.log(0.95 * r_horizon(a)), 0.0, 0.0], xmax=[math.log(1000.0), 1.0, 2.0 * math.pi],
                        bc=[BC_OUTFLOW, BC_OUTFLOW, BC_POLAR, BC_POLAR, BC_PERIODIC, BC_PERIODIC])
    elif cfg == 5:  # throughput sweep: Minkowski periodic cube, gamma = 5/3
        n1, n2, n3 = res((128, 128, 128))
        p = base_params(n1=n1, n2=n2, n3=n3, gamma=5.0 / 3.0, recon=RECON_MC)
    else:
        raise ValueError("cfg must be 1..5")
    if recon is not None:
        p["recon"] = recon
    return p
