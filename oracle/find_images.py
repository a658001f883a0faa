"""TEST INFRASTRUCTURE, NOT THE PRODUCT: plain numpy oracle for the consumer of the deflection map described in the paper's
section 2.2.2 and Fig. 1 -- SURVEY 8(f) NEXT-3:

  "we divide each pixel in the image plane into two triangles [...] we lens each triangle into the source plane by using
   equation 13 and we check if the barycenter is inside this triangle in the source plane.  If it is, a predicted
   multiple image location in the image plane is found."

Step by step, in fp64, one source point at a time, every triangle of the grid (brute force):
  1. node positions theta_ij = (x_min + i*dx, y_min + j*dx) (as the map defines them) and their source-plane images
     beta_ij = theta_ij - (D_LS/D_OS) * gradPsi_ij                                        (eq. 13)
  2. every cell (i, j), 0 <= i < nx-1, 0 <= j < ny-1, between four neighbouring nodes is cut along the diagonal from node
     (i+1, j) to node (i, j+1) into T0 = [(i,j), (i+1,j), (i,j+1)] and T1 = [(i+1,j+1), (i,j+1), (i+1,j)]   (reading R23:
     Fig. 1 shows the cut only as a picture)
  3. point-in-triangle in the source plane with the three edge functions
         e0 = (B-A) x (P-A),  e1 = (C-B) x (P-B),  e2 = (A-C) x (P-C)        (u x v = u_x v_y - u_y v_x)
     inside  <=>  all three >= 0 or all three <= 0, and e0 + e1 + e2 != 0 (reading R24: closed triangles, a point on a
     shared edge is reported by both neighbours, zero-area triangles contain nothing)
  4. the predicted image position is the image-plane point with the same barycentric coordinates,
     w_A = e1/area, w_B = e2/area, w_C = e0/area, area = e0 + e1 + e2  (reading R25: the paper only says a location
     "is found"; linear interpolation inside the triangle is exact for a locally linear lens mapping).
Imports nothing from paper_1902_03252_b200.  Only tests/ may import it.
"""
import numpy as np


def source_plane(grad, x_min, y_min, dx, dls_dos):
    """beta [ny, nx, 2] from the gradient map [ny, nx, 2] (eq. 13)."""
    g = np.asarray(grad, dtype=np.float64)
    ny, nx = g.shape[0], g.shape[1]
    t1 = x_min + np.arange(nx, dtype=np.float64) * dx
    t2 = y_min + np.arange(ny, dtype=np.float64) * dx
    beta = np.empty_like(g)
    beta[:, :, 0] = t1[None, :] - dls_dos * g[:, :, 0]
    beta[:, :, 1] = t2[:, None] - dls_dos * g[:, :, 1]
    return beta, t1, t2


def _edges(A, B, C, P):
    e0 = (B[0] - A[0]) * (P[1] - A[1]) - (B[1] - A[1]) * (P[0] - A[0])
    e1 = (C[0] - B[0]) * (P[1] - B[1]) - (C[1] - B[1]) * (P[0] - B[0])
    e2 = (A[0] - C[0]) * (P[1] - C[1]) - (A[1] - C[1]) * (P[0] - C[0])
    return e0, e1, e2


def find_images(grad, x_min, y_min, dx, dls_dos, sources):
    """All (source k, cell j*nx+i, triangle t, x, y) with source k inside the source-plane image of triangle t of cell
    (i, j); returned as a structured array sorted by (source, cell, triangle)."""
    beta, t1, t2 = source_plane(grad, x_min, y_min, dx, dls_dos)
    ny, nx = beta.shape[0], beta.shape[1]
    bx, by = beta[:, :, 0], beta[:, :, 1]
    T1, T2 = np.meshgrid(t1, t2)                       # node positions [ny, nx]
    # corner views of every cell: 00 = (i,j), 10 = (i+1,j), 01 = (i,j+1), 11 = (i+1,j+1)
    c = {"00": (slice(0, ny - 1), slice(0, nx - 1)), "10": (slice(0, ny - 1), slice(1, nx)),
         "01": (slice(1, ny), slice(0, nx - 1)), "11": (slice(1, ny), slice(1, nx))}
    tri = (("00", "10", "01"), ("11", "01", "10"))
    out = []
    for k, P in enumerate(np.asarray(sources, dtype=np.float64).reshape(-1, 2)):
        for t, (a, b, cc) in enumerate(tri):
            A, B, C = (bx[c[a]], by[c[a]]), (bx[c[b]], by[c[b]]), (bx[c[cc]], by[c[cc]])
            e0, e1, e2 = _edges(A, B, C, P)
            area = (e0 + e1) + e2
            inside = (((e0 >= 0) & (e1 >= 0) & (e2 >= 0)) | ((e0 <= 0) & (e1 <= 0) & (e2 <= 0))) & (area != 0)
            jj, ii = np.nonzero(inside)
            for j, i in zip(jj, ii):
                wA, wB, wC = e1[j, i] / area[j, i], e2[j, i] / area[j, i], e0[j, i] / area[j, i]
                x = (wA * T1[c[a]][j, i] + wB * T1[c[b]][j, i]) + wC * T1[c[cc]][j, i]
                y = (wA * T2[c[a]][j, i] + wB * T2[c[b]][j, i]) + wC * T2[c[cc]][j, i]
                out.append((k, int(j) * nx + int(i), t, x, y))
    arr = np.array(out, dtype=[("source", "i4"), ("cell", "i4"), ("triangle", "i4"), ("x", "f8"), ("y", "f8")])
    return np.sort(arr, order=["source", "cell", "triangle"])
