"""paper_2301_04835_b200 -- thin Python binding of libpsg.so (include/psg.h).

The per-MD-step enhanced-sampling hot path of PySAGES (arXiv 2301.04835), batched over
replicas, as hand-written sm_100a CUDA kernels behind a C ABI.  This package only marshals
arguments (ctypes): every step of the path runs in the kernels.  PyTorch is used for device
memory and streams, nothing else.  There is no CPU fallback: if libpsg.so is missing or no
CUDA device is present, calls raise.
"""
from .psg import (Context, PsgError, load_library, lib_path, measure_alu_peak, configure_from_workload, range_rgyr_static,
                  CV_DISTANCE, CV_ANGLE, CV_DIHEDRAL, CV_COM_COMPONENT, CV_RGYR, CV_DISPLACEMENT,
                  CV_PRINCIPAL_MOMENT, CV_ASPHERICITY, CV_ACYLINDRICITY, CV_SHAPE_ANISOTROPY, CV_DIST_TO_INTERFACE,
                  HILLS_F32, HILLS_F64, METHOD_NONE, METHOD_HARMONIC, METHOD_METAD, METHOD_ABF, METHOD_METAD_GRID, EXPORTS)

__all__ = ["Context", "PsgError", "load_library", "lib_path", "measure_alu_peak", "configure_from_workload", "range_rgyr_static",
           "CV_DISTANCE", "CV_ANGLE", "CV_DIHEDRAL", "CV_COM_COMPONENT", "CV_RGYR", "CV_DISPLACEMENT", "CV_PRINCIPAL_MOMENT",
           "CV_ASPHERICITY", "CV_ACYLINDRICITY", "CV_SHAPE_ANISOTROPY", "CV_DIST_TO_INTERFACE", "HILLS_F32", "HILLS_F64",
           "METHOD_NONE", "METHOD_HARMONIC", "METHOD_METAD", "METHOD_ABF", "METHOD_METAD_GRID", "EXPORTS"]
