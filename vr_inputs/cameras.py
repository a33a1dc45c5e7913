"""Camera recipes (BASELINE.json configs).

A camera is a plain dict: eye/right/up/forward (float32[3], orthonormal,
voxel-index world space), projection (0 perspective, 1 ortho), tan_half_fovy,
ortho_half_height.  Bases are computed in float64 and rounded once.
"""
import math

import numpy as np

PERSPECTIVE, ORTHO = 0, 1


def _cam(eye, right, up, forward, projection, tan_half_fovy=0.0, ortho_half_height=0.0):
    f32 = lambda v: np.asarray(v, dtype=np.float64).astype(np.float32)
    return {"eye": f32(eye), "right": f32(right), "up": f32(up), "forward": f32(forward),
            "projection": int(projection),
            "tan_half_fovy": float(np.float32(tan_half_fovy)),
            "ortho_half_height": float(np.float32(ortho_half_height))}


def _basis(forward, up_world=(0.0, 1.0, 0.0)):
    f = np.asarray(forward, dtype=np.float64)
    f = f / np.linalg.norm(f)
    r = np.cross(np.asarray(up_world, dtype=np.float64), f)
    r = r / np.linalg.norm(r)
    u = np.cross(f, r)
    return r, u, f


def ortho_axis_camera(dims, axis=2, half_height=None, back_off=0.5):
    """Orthographic view along +axis, eye one half-extent in front of the cube."""
    n = np.asarray(dims, dtype=np.float64)
    c = (n - 1.0) / 2.0
    f = np.zeros(3)
    f[axis] = 1.0
    up_world = (0.0, 1.0, 0.0) if axis != 1 else (0.0, 0.0, 1.0)
    r, u, f = _basis(f, up_world)
    eye = c - f * ((n[axis] - 1.0) * (0.5 + back_off) + 0.5)
    if half_height is None:
        half_height = float(np.max(np.abs(u) * (n - 1.0))) / 2.0
    return _cam(eye, r, u, f, ORTHO, ortho_half_height=half_height)


def rotate_about_y(cam, centre, degrees, half_height=None):
    """The same camera rotated about the y axis through `centre`."""
    a = math.radians(degrees)
    R = np.array([[math.cos(a), 0.0, math.sin(a)], [0.0, 1.0, 0.0],
                  [-math.sin(a), 0.0, math.cos(a)]])
    c = np.asarray(centre, dtype=np.float64)
    rot = lambda v: R @ np.asarray(v, dtype=np.float64)
    eye = c + rot(np.asarray(cam["eye"], dtype=np.float64) - c)
    hh = cam["ortho_half_height"] if half_height is None else half_height
    return _cam(eye, rot(cam["right"]), rot(cam["up"]), rot(cam["forward"]), cam["projection"],
                cam["tan_half_fovy"], hh)


def config0_views():
    """configs[0]: ortho along the frequency axis (every ray crosses 63 voxels)
    and the same camera rotated 30 degrees about y, half-height 48."""
    v1 = _cam((31.5, 31.5, -32.0), (1, 0, 0), (0, 1, 0), (0, 0, 1), ORTHO,
              ortho_half_height=31.5)
    v2 = rotate_about_y(v1, (31.5, 31.5, 31.5), 30.0, half_height=48.0)
    return [v1, v2]


def orbit_camera(dims, azimuth_deg, elevation_deg=20.0, fovy_deg=40.0, fit=0.6):
    """Perspective orbit view: eye on a sphere of radius fit*r/sin(fovy/2) around the
    cube centre, r = half the cube diagonal; look at the centre; up = +y."""
    n = np.asarray(dims, dtype=np.float64)
    c = (n - 1.0) / 2.0
    r = 0.5 * float(np.linalg.norm(n - 1.0))
    R = fit * r / math.sin(math.radians(fovy_deg / 2.0))
    az, el = math.radians(azimuth_deg), math.radians(elevation_deg)
    offs = np.array([math.cos(el) * math.sin(az), math.sin(el), -math.cos(el) * math.cos(az)])
    eye = c + R * offs
    rr, uu, ff = _basis(c - eye)
    return _cam(eye, rr, uu, ff, PERSPECTIVE,
                tan_half_fovy=math.tan(math.radians(fovy_deg / 2.0)))


def orbit_views(dims, n_views=8):
    return [orbit_camera(dims, 360.0 * k / n_views) for k in range(n_views)]
