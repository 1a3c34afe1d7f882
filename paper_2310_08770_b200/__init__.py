"""placeholder (binding added with the CUDA library)"""
