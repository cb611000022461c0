"""Ray-cast validator of the navigator (PAPER.md:49 and Fig. 1): an eta-phi picture of the
barrel (or a y-z picture of the calorimeter) taken with the transport path's own navigation calls, once with
the BVH navigator and once with the loop over all daughters; the two pictures must be identical, pixel for
pixel.  Headless: the picture goes to a PPM file.

  python -m paper_2209_15445_b200.raycast [--geometry barrel|calorimeter] [--size 1024x512] [--out picture.ppm] [--skip-loop] [--fp32]

--fp32 also takes the picture through the single-precision copy of the geometry and reports how it differs from
the fp64 picture and the ratio of the two ray rates.
"""
import argparse
import time

import numpy as np

from .inputs import field, geometry, materials


def barrel_rays(width, height, eta_max=1.45):
    """Pinhole at the origin: column = phi in [0, 2 pi), row = eta in (-eta_max, eta_max), pixel centres."""
    phi = (np.arange(width) + 0.5) * (2.0 * np.pi / width)
    eta = -eta_max + (np.arange(height) + 0.5) * (2.0 * eta_max / height)
    theta = 2.0 * np.arctan(np.exp(-eta))
    d = np.stack([np.outer(np.sin(theta), np.cos(phi)), np.outer(np.sin(theta), np.sin(phi)),
                  np.outer(np.cos(theta), np.ones(width))], axis=-1).reshape(-1, 3)
    return np.zeros_like(d), d


def calorimeter_rays(width, height, half=25.0):
    """Parallel rays along +x from the plane x = -10: column = y, row = z, pixel centres in (-half, half)."""
    y = -half + (np.arange(width) + 0.5) * (2.0 * half / width)
    z = -half + (np.arange(height) + 0.5) * (2.0 * half / height)
    p = np.stack([np.full((height, width), -10.0), np.tile(y, (height, 1)), np.tile(z[:, None], (1, width))], axis=-1).reshape(-1, 3)
    d = np.zeros_like(p)
    d[:, 0] = 1.0
    return p, d


def write_ppm(path, column, width, height):
    """Column density as a grey-scale P6 picture (white = most material)."""
    v = column.reshape(height, width)
    top = v.max() if v.max() > 0 else 1.0
    g = np.clip(255.0 * v / top, 0, 255).astype(np.uint8)
    with open(path, "wb") as f:
        f.write(f"P6\n{width} {height}\n255\n".encode())
        f.write(np.repeat(g[:, :, None], 3, axis=2).tobytes())


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--geometry", default="barrel", choices=["barrel", "calorimeter"])
    ap.add_argument("--size", default="1024x512")
    ap.add_argument("--out", default="")
    ap.add_argument("--skip-loop", action="store_true", help="BVH picture only (the loop navigator tests 61 200 crystals per step)")
    ap.add_argument("--fp32", action="store_true", help="also the single-precision geometry mode (BVH navigator)")
    args = ap.parse_args()
    from . import adept
    w, h = (int(x) for x in args.size.split("x"))
    g = geometry.barrel() if args.geometry == "barrel" else geometry.calorimeter()
    _, tabs, scal = materials.build_material_set(g.material_names)
    pos, d = barrel_rays(w, h) if args.geometry == "barrel" else calorimeter_rays(w, h)
    a = adept.Adept(g, tabs, scal, field.no_field(), track_capacity=1 << 10)
    res, rate = {}, {}
    for name, nav in (("bvh", adept.NAV_BVH), ("loop", adept.NAV_LOOP), ("bvh_fp32", adept.NAV_BVH_F32)):
        if (nav == adept.NAV_LOOP and args.skip_loop) or (nav == adept.NAV_BVH_F32 and not args.fp32):
            continue
        a.raycast(pos[:1024], d[:1024], nav)          # warm-up
        t0 = time.perf_counter()
        col, nx, ms = a.raycast(pos, d, nav)
        res[name] = (col, nx)
        rate[name] = len(col) / ms * 1e3
        print(f"{name}: {len(col)} rays, {int(nx.sum())} boundary crossings, kernel {ms:.2f} ms = {len(col) / ms * 1e3:.3e} rays/s, "
              f"{nx.sum() / ms * 1e3:.3e} crossings/s (host call {1e3 * (time.perf_counter() - t0):.1f} ms)")
    if "bvh_fp32" in res:
        c64, n64 = res["bvh"]
        c32, n32 = res["bvh_fp32"]
        same_nx = n32 == n64
        rel = np.abs(c32[same_nx] - c64[same_nx]) / np.maximum(c64[same_nx], 1e-30)
        print(f"fp32 vs fp64 picture: {100.0 * same_nx.mean():.3f} % of the rays cross the same number of boundaries; column density of those "
              f"differs by at most {rel.max():.2e} relative; fp32 / fp64 ray rate {rate['bvh_fp32'] / rate['bvh']:.2f}")
    if "loop" in res:
        same = np.array_equal(res["bvh"][1], res["loop"][1]) and np.array_equal(res["bvh"][0], res["loop"][0])
        print("BVH picture == loop picture, bit for bit:", same)
    if args.out:
        write_ppm(args.out, res["bvh"][0], w, h)
        print("wrote", args.out)
    a.close()


if __name__ == "__main__":
    main()
